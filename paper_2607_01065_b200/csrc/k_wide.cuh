// k_wide.cuh -- the paper's own operating points: wide sub-vectors d = 64 / 128 / 256 (D = 128 with
// R = 32 / 16 / 12 stages, D = 256 with R = 12; K = 256), and the textbook weighted K-means (KM) baseline of the Fig. 4
// comparison (PAPER.md:60-85 section 4, :202-212) with up to 4096 centroids.  These kernels are exact by construction:
//   k_wide_prep     gather the fit rows (warp per row), row norms in fp64, weights, bf16 operand planes for the
//                   tensor-core filter (k_score_tc_wide.cuh)
//   k_wide_init     seeded initial rows (Alg. 1 l.1; reading c-I), any d
//   k_wide_assign   arg-max of Eq. 5 (or the plain projection, or the KM distance) in fp64 with the definition's own
//                   operation order, for all rows or for the rows a filter could not decide
//   k_wide_update   weighted cluster sums in fp64 in ascending row order (one CTA per cluster), Eq. 7 / Eq. 8 with the
//                   safeguards of PAPER.md:178, or the KM centroid (weighted mean)
//   k_wide_subtract r <- fl32(r - fl32(g_k s_k)) and the code byte (RQ); operand planes of the new residual
//   k_wide_decode   xhat = sum of the stages' codewords in fp32 stage order (reading c-D)
// No floating-point atomics; every sum has a fixed order.
#pragma once
#include "gsrq_common.cuh"

namespace gsrq {
namespace wide {

constexpr int kMaxD = 256;
constexpr int kMaxK = 4096;

enum { kModeGskm = 0, kModeProj = 1, kModeKm = 2 };   // scoring rule of k_wide_assign

// ---------------------------------------------------------------------------------------------------- prep
struct WPrepParams {
  RowSrc src;                  // kv (strided, bf16 / fp32) or fp32 rows [G][rows_per_group][d]
  const float *w;              // [.][T] per-token weights or nullptr
  long long w_stride_g;
  const long long *fit_tokens; // [G][nf_tok] or nullptr
  long long nf_tok;
  float *Rf;                   // [G][Nf][d] compact fp32 rows (out; may alias src.rows when there is no gather)
  float *wt;                   // [G][nf_tok]
  double *wn;                  // [G][Nf] w_i / (||r_i|| + eps)
  float *rnorm;                // [G][Nf] upper bound of ||r_i|| (fp32) or nullptr
  double *epart;               // [G][gridDim.x] partials of sum w_i ||r_i||^2, or nullptr
  __nv_bfloat16 *ahi, *alo;    // [G][Nf][d] bf16 operand planes or nullptr
};

// warp per row, 8 rows per CTA.  grid = (ceil(Nf / 8), G), block = 256.
__global__ void __launch_bounds__(256) k_wide_prep(WPrepParams p) {
  __shared__ double esh[8];
  const int g = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int d = p.src.d;
  const long long Nf = p.nf_tok * p.src.M;
  const long long i = (long long)blockIdx.x * 8 + warp;
  double e = 0.0;
  if (i < Nf) {
    const long long tl = i / p.src.M;
    const int m = (int)(i - tl * p.src.M);
    const long long tok = p.fit_tokens ? p.fit_tokens[(long long)g * p.nf_tok + tl] : tl;
    const long long gi = (long long)g * Nf + i;
    double n2 = 0.0;
    for (int e0 = lane * 4; e0 < d; e0 += 128) {
      float x[4];
      if (p.src.rows) {
        const float4 v = *reinterpret_cast<const float4 *>(p.src.rows + ((long long)g * p.src.rows_per_group + tok * p.src.M + m) * d + e0);
        x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
      } else if (p.src.dtype == GSRQ_BF16) {
        const uint2 v = *reinterpret_cast<const uint2 *>(reinterpret_cast<const uint16_t *>(p.src.kv) + (long long)g * p.src.stride_g + tok * p.src.stride_t + (long long)m * d + e0);
        x[0] = __uint_as_float(v.x << 16); x[1] = __uint_as_float(v.x & 0xFFFF0000u);
        x[2] = __uint_as_float(v.y << 16); x[3] = __uint_as_float(v.y & 0xFFFF0000u);
      } else {
        const float4 v = *reinterpret_cast<const float4 *>(reinterpret_cast<const float *>(p.src.kv) + (long long)g * p.src.stride_g + tok * p.src.stride_t + (long long)m * d + e0);
        x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
      }
      *reinterpret_cast<float4 *>(p.Rf + gi * d + e0) = make_float4(x[0], x[1], x[2], x[3]);
#pragma unroll
      for (int u = 0; u < 4; ++u) n2 = __dadd_rn(n2, __dmul_rn((double)x[u], (double)x[u]));
      if (p.ahi) {
        uint32_t h[2], l[2];
#pragma unroll
        for (int u = 0; u < 4; u += 2) {
          const __nv_bfloat16 h0 = __float2bfloat16_rn(x[u]), h1 = __float2bfloat16_rn(x[u + 1]);
          const __nv_bfloat16 l0 = __float2bfloat16_rn(__fsub_rn(x[u], __bfloat162float(h0)));
          const __nv_bfloat16 l1 = __float2bfloat16_rn(__fsub_rn(x[u + 1], __bfloat162float(h1)));
          h[u / 2] = (uint32_t)__bfloat16_as_ushort(h0) | ((uint32_t)__bfloat16_as_ushort(h1) << 16);
          l[u / 2] = (uint32_t)__bfloat16_as_ushort(l0) | ((uint32_t)__bfloat16_as_ushort(l1) << 16);
        }
        *reinterpret_cast<uint2 *>(p.ahi + gi * d + e0) = make_uint2(h[0], h[1]);
        if (p.alo) *reinterpret_cast<uint2 *>(p.alo + gi * d + e0) = make_uint2(l[0], l[1]);
      }
    }
    for (int off = 16; off; off >>= 1) n2 += __shfl_xor_sync(0xffffffffu, n2, off);   // fixed tree: every lane ends with the same sum
    const double n = sqrt(n2);
    const float wv = p.w ? p.w[(long long)g * p.w_stride_g + tok] : 1.0f;
    if (lane == 0) {
      if (m == 0) p.wt[(long long)g * p.nf_tok + tl] = wv;
      p.wn[gi] = (double)wv * (1.0 / (n + kEps));
      if (p.rnorm) p.rnorm[gi] = (float)n * 1.000001f;
    }
    e = (double)wv * n2;
  }
  if (!p.epart) return;
  if (lane == 0) esh[warp] = e;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int q = 0; q < 8; ++q) s += esh[q];
    p.epart[(long long)g * gridDim.x + blockIdx.x] = s;
  }
}

// ---------------------------------------------------------------------------------------------------- init
// Same candidate stream and acceptance rule as k_init_ids (k_prep.cuh), for any d.  grid = G, block = 512.
// shapes == nullptr: ids only.  km: the initial centroids are the chosen rows themselves (not normalised), gains = 1.
__global__ void __launch_bounds__(512) k_wide_init(const float *__restrict__ Rf, long long Nf, int d, int K, int G, int stage,
                                                   uint64_t seed, long long *__restrict__ ids, DevStats *__restrict__ st,
                                                   float *__restrict__ shapes, float *__restrict__ gains, long long cb_stride_g, int km) {
  __shared__ long long cand[512];
  __shared__ int ok[512];
  __shared__ int scan[512];
  __shared__ int n_chosen;
  extern __shared__ long long chosen[];   // [K]
  const int g = blockIdx.x, t = threadIdx.x;
  const uint64_t sg = seed ^ (kGamma * (uint64_t)(1 + g + G * stage));
  if (t == 0) n_chosen = 0;
  __syncthreads();
  const long long limit = 64LL * K + 4096;
  for (long long base = 0; base < limit; base += 512) {
    const long long n = base + t;
    const long long c = (long long)(splitmix64_at(sg, (uint64_t)n) % (uint64_t)Nf);
    int good = n < limit;
    if (good) {
      const float *x = Rf + ((long long)g * Nf + c) * d;
      bool nz = false;
      for (int j = 0; j < d; ++j) nz |= (x[j] != 0.0f);
      good = nz;
    }
    cand[t] = c;
    __syncthreads();
    const int nc = n_chosen;
    if (good) {
      int dup = 0;
      for (int q = 0; q < nc; ++q) dup |= (chosen[q] == c);
      for (int q = 0; q < t; ++q) dup |= (cand[q] == c);
      good = !dup;
    }
    ok[t] = good;
    scan[t] = good;
    __syncthreads();
    for (int off = 1; off < 512; off <<= 1) {
      const int v = (t >= off) ? scan[t - off] : 0;
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
  const bool degenerate = n_chosen < K;
  if (degenerate && t == 0) st[g].err = GSRQ_EDEGENERATE;
  for (int k = t; k < K; k += 512) ids[(long long)g * K + k] = (k < n_chosen) ? chosen[k] : 0;
  if (!shapes) return;
  for (int k = t; k < K; k += 512) {
    const float *x = Rf + ((long long)g * Nf + (k < n_chosen ? chosen[k] : 0)) * d;
    float *s = shapes + ((long long)g * cb_stride_g + k) * d;
    double n2 = 0.0;
    for (int j = 0; j < d; ++j) n2 = __dadd_rn(n2, __dmul_rn((double)x[j], (double)x[j]));
    const double n = sqrt(n2);
    for (int j = 0; j < d; ++j) s[j] = km ? x[j] : ((n > 0.0) ? (float)((double)x[j] / n) : 0.0f);
    gains[(long long)g * cb_stride_g + k] = km ? 1.0f : 0.0f;
  }
}

// ---------------------------------------------------------------------------------------------------- assign
struct WAssignParams {
  const float *rows;      // [G][N][d] fp32
  long long N;
  int d, K, mode;         // kModeGskm / kModeProj / kModeKm
  const float *shapes;    // stage slice: codeword k of group g at shapes + (g*cb_stride_g + k)*d   (KM: the centroid itself)
  const float *gains;
  long long cb_stride_g;
  void *idx;              // [G][N] uint8 (idx16 == 0) or uint16
  int idx16;
  const uint32_t *list;   // rows to score: {g*N + i}, or nullptr = every row
  const unsigned int *list_cnt;
  DevStats *st;           // changed[slot] += rows whose assignment changed (nullptr: not counted)
  int slot;
  double *best_out;       // optional [G][N] best score (tests)
};

constexpr int kWaRows = 32, kWaCw = 32;   // tile: 32 rows x chunks of 32 codewords; block = 256

__host__ __device__ inline size_t wide_assign_smem(int d) { return ((size_t)kWaRows * (d + 1) + (size_t)kWaCw * d) * sizeof(double) + kWaRows * 8 * 16; }

// Exact arg-max, the oracle's arithmetic: dot = sum_j x_j s_kj in element order, products and sums rounded separately
// (no FMA contraction); score = (2 g) dot - g g; lowest k wins ties (reading c-T).  KM: dist = sum_j (x_j - mu_kj)^2 in
// element order, arg-MIN, lowest k on ties.  Thread (r = tid % 32, q = tid / 32) scores row r against codewords
// 4 q .. 4 q + 3 of every 32-codeword chunk (ascending k), then the 8 threads of a row are merged in ascending q.
// grid = (ceil(n_rows / 32), G or 1 with a list), block = 256, dynamic smem = wide_assign_smem(d).
__global__ void __launch_bounds__(256) k_wide_assign(WAssignParams p) {
  extern __shared__ __align__(16) double wsm[];
  const int d = p.d;
  double *xs = wsm;                       // [32][d + 1]
  double *cw = xs + kWaRows * (d + 1);    // [32][d]
  double *mb = cw + kWaCw * d;            // [32][8] best scores
  int *mk = reinterpret_cast<int *>(mb + kWaRows * 8);   // [32][8] best indices
  const int tid = threadIdx.x, r = tid & 31, q = tid >> 5;
  long long n_rows = p.N;
  const int g_blk = blockIdx.y;
  if (p.list) n_rows = (long long)*p.list_cnt;
  else if (group_done(p.st, g_blk, p.slot)) return;
  for (long long t0 = (long long)blockIdx.x * kWaRows; t0 < n_rows; t0 += (long long)gridDim.x * kWaRows) {
    int g = g_blk;
    // global row of my tile row (list mode: rows of any group)
    long long grow = -1;
    if (t0 + r < n_rows) grow = p.list ? (long long)p.list[t0 + r] : (long long)g * p.N + t0 + r;
    __syncthreads();   // the previous tile is done with the shared buffers
    // stage the tile's rows as fp64: warp q converts rows q, q + 8, ...
    for (int rr = q; rr < kWaRows; rr += 8) {
      const long long gr = (t0 + rr < n_rows) ? (p.list ? (long long)p.list[t0 + rr] : (long long)g * p.N + t0 + rr) : -1;
      for (int j = r; j < d; j += 32) xs[rr * (d + 1) + j] = (gr >= 0) ? (double)p.rows[gr * d + j] : 0.0;
    }
    const int my_g = (grow >= 0) ? (int)(grow / p.N) : 0;   // list mode: the row's group
    // list mode can mix groups in one tile: the codeword chunk in shared memory is only used when the whole tile is one group
    bool uniform = !p.list;
    if (p.list) {
      const int g0 = (int)((long long)p.list[t0] / p.N);
      const int same = __syncthreads_and((grow < 0) || (my_g == g0));
      uniform = same != 0;
      g = g0;
    }
    double best = (p.mode == kModeKm) ? INFINITY : -INFINITY;
    int bk = 0x7fffffff;
    __syncthreads();
    for (int k0 = 0; k0 < p.K; k0 += kWaCw) {
      if (uniform) {
        __syncthreads();
        for (int e = tid; e < kWaCw * d; e += 256) {
          const int kk = k0 + e / d;
          cw[e] = (kk < p.K) ? (double)p.shapes[((long long)g * p.cb_stride_g + kk) * d + (e % d)] : 0.0;
        }
        __syncthreads();
      }
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
      const double *xr = xs + r * (d + 1);
      if (uniform) {
        const double *c0 = cw + (4 * q) * d;
        for (int j = 0; j < d; ++j) {
          const double x = xr[j];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const double c = c0[u * d + j];
            if (p.mode == kModeKm) { const double e = __dsub_rn(x, c); acc[u] = __dadd_rn(acc[u], __dmul_rn(e, e)); }
            else acc[u] = __dadd_rn(acc[u], __dmul_rn(x, c));
          }
        }
      } else if (grow >= 0) {
        for (int u = 0; u < 4; ++u) {
          const int kk = k0 + 4 * q + u;
          if (kk >= p.K) break;
          const float *c0 = p.shapes + ((long long)my_g * p.cb_stride_g + kk) * d;
          double a = 0.0;
          for (int j = 0; j < d; ++j) {
            const double x = xr[j], c = (double)c0[j];
            if (p.mode == kModeKm) { const double e = __dsub_rn(x, c); a = __dadd_rn(a, __dmul_rn(e, e)); }
            else a = __dadd_rn(a, __dmul_rn(x, c));
          }
          acc[u] = a;
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int kk = k0 + 4 * q + u;
        if (kk >= p.K) continue;
        double sc = acc[u];
        if (p.mode == kModeGskm) {
          const double gk = (double)p.gains[(long long)(uniform ? g : my_g) * p.cb_stride_g + kk];
          sc = __dsub_rn(__dmul_rn(__dmul_rn(2.0, gk), acc[u]), __dmul_rn(gk, gk));
        }
        const bool better = (p.mode == kModeKm) ? (sc < best) : (sc > best);
        if (better) { best = sc; bk = kk; }   // ascending k within the thread: strict comparison keeps the lowest index
      }
    }
    mb[r * 8 + q] = best;
    mk[r * 8 + q] = bk;
    __syncthreads();
    if (q == 0 && grow >= 0) {
      double b = mb[r * 8];
      int k = mk[r * 8];
      for (int u = 1; u < 8; ++u) {
        const double ob = mb[r * 8 + u];
        const int ok_ = mk[r * 8 + u];
        const bool better = (p.mode == kModeKm) ? (ob < b) : (ob > b);
        if (better || (ob == b && ok_ < k)) { b = ob; k = ok_; }
      }
      if (k == 0x7fffffff) k = 0;
      int old;
      if (p.idx16) { uint16_t *ip = reinterpret_cast<uint16_t *>(p.idx) + grow; old = *ip; *ip = (uint16_t)k; }
      else { uint8_t *ip = reinterpret_cast<uint8_t *>(p.idx) + grow; old = *ip; *ip = (uint8_t)k; }
      if (p.best_out) p.best_out[grow] = b;
      if (p.st && old != k) atomicAdd(reinterpret_cast<unsigned long long *>(&p.st[(int)(grow / p.N)].changed[p.slot]), 1ull);
    }
  }
}

// The rows the tensor-core filter could not decide: list entry {g*N + i, mask of the 16-codeword groups whose filter maximum lies
// within the decision margin} -- a codeword outside those groups cannot be the exact arg-max.  One warp per
// entry: the row is staged in shared memory as fp64, lane l scores codeword 16 c + l % 16 of two candidate groups per round with
// the oracle's arithmetic (element order, separate multiply and add), lowest k wins ties.  grid-stride; block = 256 (8 warps),
// dynamic smem = 8 * d * 8 bytes.
__global__ void __launch_bounds__(256) k_wide_refine(WAssignParams p, const uint2 *__restrict__ list2) {
  extern __shared__ __align__(16) double rsm[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, d = p.d;
  double *xs = rsm + warp * d;
  const unsigned int n = *p.list_cnt;
  for (unsigned int e = blockIdx.x * 8 + warp; e < n; e += gridDim.x * 8) {
    const uint2 en = list2[e];
    const long long grow = en.x;
    const int g = (int)(grow / p.N);
    uint32_t gmask = en.y & 0xFFFFu;
    __syncwarp();
    for (int j = lane; j < d; j += 32) xs[j] = (double)p.rows[grow * d + j];
    __syncwarp();
    double best = -INFINITY;
    int bi = 0x7fffffff;
    while (gmask) {
      const int c0 = __ffs(gmask) - 1;
      gmask &= gmask - 1;
      int c1 = -1;
      if (gmask) { c1 = __ffs(gmask) - 1; gmask &= gmask - 1; }
      const int c = (lane < 16) ? c0 : c1;
      const int kk = 16 * c + (lane & 15);
      if (c >= 0 && kk < p.K) {
        const float *sk = p.shapes + ((long long)g * p.cb_stride_g + kk) * d;
        double dot = 0.0;
        for (int j = 0; j < d; j += 4) {
          const float4 sv = __ldg(reinterpret_cast<const float4 *>(sk + j));
          dot = __dadd_rn(dot, __dmul_rn(xs[j], (double)sv.x));
          dot = __dadd_rn(dot, __dmul_rn(xs[j + 1], (double)sv.y));
          dot = __dadd_rn(dot, __dmul_rn(xs[j + 2], (double)sv.z));
          dot = __dadd_rn(dot, __dmul_rn(xs[j + 3], (double)sv.w));
        }
        double sc = dot;
        if (p.mode == kModeGskm) {
          const double gk = (double)p.gains[(long long)g * p.cb_stride_g + kk];
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
    if (lane == 0) {
      const int k = (bi == 0x7fffffff) ? 0 : bi;
      uint8_t *ip = reinterpret_cast<uint8_t *>(p.idx) + grow;
      const int old = *ip;
      *ip = (uint8_t)k;
      if (p.st && old != k) atomicAdd(reinterpret_cast<unsigned long long *>(&p.st[g].changed[p.slot]), 1ull);
    }
  }
}

// ---------------------------------------------------------------------------------------------------- update
struct WUpdateParams {
  const float *rows;      // [G][N][d]
  const double *wn;       // [G][N]
  const float *wt;        // [G][nf_tok]
  long long nf_tok;
  int M;
  const void *idx;        // [G][N] uint8 / uint16
  int idx16;
  long long N;
  int d, K;
  float *shapes, *gains;  // stage slice
  long long cb_stride_g;
  int mode;               // 0: gains only (Alg. 1 l.2); 1: shapes + gains (Eq. 7, Eq. 8); 2: KM centroid = weighted mean
  DevStats *st;           // or nullptr
  double *term;           // [G][term_stride][term_k] per-cluster terms of J, or nullptr
  int term_stride, term_k;
  int t;
  int *gmax;              // optional [G]: bit pattern of max_k g_k after this update (atomicMax on an int), for the tensor-core filter
  int nparts;             // the rows of a group are split in nparts contiguous ranges (gridDim.z), one CTA each
  double *part;           // nparts > 1: [G][K][nparts][2d + 2] partial sums, merged in range order by k_wide_update_finish
  // sorted mode (K <= 256, uint8 assignment; k_wide_bucket -> k_wide_items -> k_wide_update_items -> k_wide_update_items_finish):
  const int *order;       // [G][N] row indices, sub-range by sub-range, cluster by cluster, ascending (stable counting sort)
  const int *starts;      // [G][nsub][K + 1] first position of each cluster within its sub-range's part of order
  int nsub;               // <= 32
  int *item_first;        // [G][K + 1] first work item of each cluster; an item = up to kItemRows consecutive rows of one cluster's list
  int max_items;          // bound of the items of a group: N / kItemRows + K; part is [G][max_items][2d + 2] in this mode
};

constexpr int kMaxSub = 32;      // sub-ranges per group in sorted mode (one per lane in k_wide_update_items)
constexpr int kItemRows = 64;
inline size_t wide_update_smem() { return (size_t)2048 * 16; }
// first row of sub-range sp of nsub (16-row aligned; sub-range nsub starts at N)
__host__ __device__ inline long long wide_sub_begin(long long N, int sp, int nsub) { return sp >= nsub ? N : ((N * (long long)sp / nsub) & ~15LL); }

// Stable counting sort of the rows of one sub-range by cluster.  Thread t owns the rows [t per, (t + 1) per) of the sub-range and its
// own row of a [256][K] table of uint16 counters: count, exclusive scan over (cluster, thread), scatter.  Rows of a cluster come
// out in ascending order.  grid = (nsub, G), block = 256, dynamic shared memory 256 K uint16.
struct WBucketParams {
  const uint8_t *idx;     // [G][N]
  long long N;
  int K, nsub;
  int *order, *starts;
  const DevStats *st;
  int t;
};

__global__ void __launch_bounds__(256) k_wide_bucket(WBucketParams p) {
  extern __shared__ __align__(16) uint16_t btab[];   // [256][K]
  __shared__ int start[257];
  __shared__ int wtot[8];
  const int sp = blockIdx.x, g = blockIdx.y, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, K = p.K;
  if (group_done(p.st, g, p.t)) return;
  const long long rb = wide_sub_begin(p.N, sp, p.nsub), re = wide_sub_begin(p.N, sp + 1, p.nsub);
  const int n = (int)(re - rb), per = (n + 255) / 256;
  const int b = min(n, tid * per), e = min(n, b + per);
  const uint8_t *ix = p.idx + (long long)g * p.N + rb;
  for (int q = tid; q < 128 * K; q += 256) reinterpret_cast<uint32_t *>(btab)[q] = 0u;
  __syncthreads();
  uint16_t *mine = btab + tid * K;
  for (int i = b; i < e; ++i) { const int k = ix[i]; if (k < K) ++mine[k]; }   // a byte >= K (caller's assignment) belongs to no cluster
  __syncthreads();
  int run = 0;
  if (tid < K)
    for (int t = 0; t < 256; ++t) { const int c = btab[t * K + tid]; btab[t * K + tid] = (uint16_t)run; run += c; }
  int incl = run;
  for (int off = 1; off < 32; off <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, off); if (lane >= off) incl += v; }
  if (lane == 31) wtot[warp] = incl;
  __syncthreads();
  int base = 0;
  for (int w8 = 0; w8 < warp; ++w8) base += wtot[w8];
  start[tid] = base + incl - run;
  if (tid == 255) start[256] = base + incl;
  __syncthreads();
  int *ord = p.order + (long long)g * p.N + rb;
  for (int i = b; i < e; ++i) {
    const int k = ix[i];
    if (k < K) ord[start[k] + (int)(mine[k]++)] = (int)(rb + i);
  }
  int *so = p.starts + ((long long)g * p.nsub + sp) * (K + 1);
  for (int k = tid; k <= K; k += 256) so[k] = start[k];
}

// Eq. 7 / Eq. 8 (or the KM centroid) for cluster k of group g from its sums fin = A[d] | B[d] | W | cnt; all 256 threads.
__device__ __forceinline__ void wide_finish_cluster(const WUpdateParams &p, int g, int k, const double *fin, double *red);

// One CTA per (cluster, group, row range): scan the range's assignment, collect the cluster's rows in ascending order, add them
// up in fp64 in that order (thread = element: A_e for e < d, B_e for the next d values); with one range per group the CTA goes
// on to Eq. 7 / Eq. 8, else the partial sums go to global memory for k_wide_update_finish (heavy-tailed cluster sizes: a
// cluster with thousands of rows would otherwise keep one CTA busy long after the others have finished).
// grid = (K, G, nparts), block = 256, dynamic shared memory wide_update_smem().  NQ = float4 per lane and row = ceil(d / 128).
template <int NQ>
__global__ void __launch_bounds__(256) k_wide_update(WUpdateParams p) {
  constexpr int kScanChunk = 2048, kChunk = kScanChunk;   // rows scanned per round (8 per thread)
  extern __shared__ __align__(16) uint8_t upd_raw[];
  double *wnq = reinterpret_cast<double *>(upd_raw);           // [kChunk] w_i / (||r_i|| + eps) of the round's matching rows, ascending
  int *rowq = reinterpret_cast<int *>(wnq + kChunk);           // their row (offset from the round's first row / index in the group)
  float *wq = reinterpret_cast<float *>(rowq + kChunk);        // their weights w_i
  __shared__ int wcnt[8];
  __shared__ double fin[2 * kMaxD + 2];
  __shared__ double red[256];
  const int k = blockIdx.x, g = blockIdx.y, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (group_done(p.st, g, p.t)) return;
  const long long rb = (p.N * (long long)blockIdx.z / p.nparts) & ~15LL;   // range starts on a 16-row boundary
  const long long re = (blockIdx.z + 1 == (unsigned)p.nparts) ? p.N : ((p.N * (long long)(blockIdx.z + 1) / p.nparts) & ~15LL);
  const int d = p.d;
  const int msh = ((p.M & (p.M - 1)) == 0) ? (31 - __clz(p.M)) : -1;
  // warp w adds the list entries w, w + 8, ... (ascending), lane l the elements 4 l .. 4 l + 3 (+ 128 q): A (coefficient w) and
  // B (coefficient w / (||r|| + eps)) of the same elements, so a row is widened to fp64 once
  double accA[NQ][4], accB[NQ][4];
#pragma unroll
  for (int q = 0; q < NQ; ++q)
#pragma unroll
    for (int j = 0; j < 4; ++j) { accA[q][j] = 0.0; accB[q][j] = 0.0; }
  double accW = 0.0;
  long long cnt = 0;
  const float *rows_g = p.rows + (long long)g * p.N * d;
  bool live[NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) live[q] = 4 * lane + 128 * q < d;
  auto add_rows = [&](const float *rows_c, int total) {
    constexpr int kDepth = 4;   // rows in flight per warp
    for (int r0 = warp; r0 < total; r0 += 8 * kDepth) {
      float4 x[kDepth][NQ];
#pragma unroll
      for (int u = 0; u < kDepth; ++u)
#pragma unroll
        for (int q = 0; q < NQ; ++q)
          x[u][q] = (r0 + 8 * u < total && live[q]) ? __ldg(reinterpret_cast<const float4 *>(rows_c + (long long)rowq[r0 + 8 * u] * d + 4 * lane + 128 * q))
                                                     : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int u = 0; u < kDepth; ++u) {
        if (r0 + 8 * u < total) {
          const double wv = (double)wq[r0 + 8 * u], wnv = wnq[r0 + 8 * u];
#pragma unroll
          for (int q = 0; q < NQ; ++q) {
            const double v[4] = {(double)x[u][q].x, (double)x[u][q].y, (double)x[u][q].z, (double)x[u][q].w};
#pragma unroll
            for (int j = 0; j < 4; ++j) { accA[q][j] = fma(wv, v[j], accA[q][j]); accB[q][j] = fma(wnv, v[j], accB[q][j]); }
          }
          if (lane == 0) accW += wv;
        }
      }
    }
    cnt += total;
  };
  for (long long c0 = rb; c0 < re; c0 += kScanChunk) {
    // ordered compaction of the matching rows of [c0, c0 + kScanChunk): thread t looks at rows c0 + 8 t .. + 7
    int my[8], nm = 0;
    const long long b0 = c0 + 8LL * tid;
    if (!p.idx16 && b0 + 8 <= re && (((long long)g * p.N + b0) & 7) == 0) {   // 8 assignment bytes in one load
      const uint2 v2 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const uint8_t *>(p.idx) + (long long)g * p.N + b0);
#pragma unroll
      for (int u = 0; u < 8; ++u) { my[u] = (int)(((u < 4 ? v2.x : v2.y) >> (8 * (u & 3))) & 255u) == k; nm += my[u]; }
    } else {
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const long long i = b0 + u;
        int v = -1;
        if (i < re) v = p.idx16 ? (int)reinterpret_cast<const uint16_t *>(p.idx)[(long long)g * p.N + i] : (int)reinterpret_cast<const uint8_t *>(p.idx)[(long long)g * p.N + i];
        my[u] = (v == k);
        nm += my[u];
      }
    }
    int incl = nm;
    for (int off = 1; off < 32; off <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, off); if (lane >= off) incl += v; }
    if (lane == 31) wcnt[warp] = incl;
    __syncthreads();
    int base = 0, total = 0;
    for (int w8 = 0; w8 < 8; ++w8) { if (w8 < warp) base += wcnt[w8]; total += wcnt[w8]; }
    int pos = base + incl - nm;
#pragma unroll
    for (int u = 0; u < 8; ++u)
      if (my[u]) {
        const long long i = b0 + u;
        rowq[pos] = (int)(i - c0);
        wq[pos] = __ldg(p.wt + (long long)g * p.nf_tok + ((msh >= 0) ? (i >> msh) : (i / p.M)));
        wnq[pos] = __ldg(p.wn + (long long)g * p.N + i);
        ++pos;
      }
    __syncthreads();
    add_rows(rows_g + c0 * d, total);
    __syncthreads();
  }
  // the eight warps' sums, added in warp order
  for (int w8 = 0; w8 < 8; ++w8) {
    if (warp == w8) {
#pragma unroll
      for (int q = 0; q < NQ; ++q)
        if (live[q])
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int e = 4 * lane + 128 * q + j;
            fin[e] = (w8 ? fin[e] : 0.0) + accA[q][j];
            fin[d + e] = (w8 ? fin[d + e] : 0.0) + accB[q][j];
          }
      if (lane == 0) fin[2 * d] = (w8 ? fin[2 * d] : 0.0) + accW;
    }
    __syncthreads();
  }
  if (tid == 0) fin[2 * d + 1] = (double)cnt;
  __syncthreads();
  if (p.nparts > 1) {
    double *out = p.part + (((long long)g * p.K + k) * p.nparts + blockIdx.z) * (2 * d + 2);
    for (int v = tid; v < 2 * d + 2; v += 256) out[v] = fin[v];
    return;
  }
  wide_finish_cluster(p, g, k, fin, red);
}

// Merge the nparts partial sums of a cluster in range order, then Eq. 7 / Eq. 8.  grid = (K, G), block = 256.
__global__ void __launch_bounds__(256) k_wide_update_finish(WUpdateParams p) {
  __shared__ double fin[2 * kMaxD + 2];
  __shared__ double red[256];
  const int k = blockIdx.x, g = blockIdx.y, tid = threadIdx.x;
  if (group_done(p.st, g, p.t)) return;
  const int d = p.d;
  const double *in = p.part + ((long long)g * p.K + k) * p.nparts * (2 * d + 2);
  for (int v = tid; v < 2 * d + 2; v += 256) {
    double sum = 0.0;
    for (int q = 0; q < p.nparts; ++q) sum += in[(long long)q * (2 * d + 2) + v];
    fin[v] = sum;
  }
  __syncthreads();
  wide_finish_cluster(p, g, k, fin, red);
}

// ---- sorted mode ----
// Work items of a group from the sorted lists: cluster k with n_k rows gets ceil(n_k / kItemRows) items.  grid = G, block = 256.
__global__ void __launch_bounds__(256) k_wide_items(WUpdateParams p) {
  __shared__ int wtot[8];
  const int g = blockIdx.x, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (group_done(p.st, g, p.t)) return;
  int n = 0;
  if (tid < p.K)
    for (int sp = 0; sp < p.nsub; ++sp) {
      const int *stp = p.starts + ((long long)g * p.nsub + sp) * (p.K + 1);
      n += stp[tid + 1] - stp[tid];
    }
  const int items = (n + kItemRows - 1) / kItemRows;
  int incl = items;
  for (int off = 1; off < 32; off <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, off); if (lane >= off) incl += v; }
  if (lane == 31) wtot[warp] = incl;
  __syncthreads();
  int base = 0;
  for (int w8 = 0; w8 < warp; ++w8) base += wtot[w8];
  int *out = p.item_first + (long long)g * (p.K + 1);
  if (tid < p.K) out[tid] = base + incl - items;
  if (tid == p.K - 1) out[p.K] = base + incl;
}

// One warp per work item: up to kItemRows rows of one cluster, added in ascending order in fp64 (lane l: the elements 4 l .. 4 l + 3
// (+ 128 q) of A and of B), eight rows in flight; the item's sums go to part[g][item].  No block-wide barrier after the table load.
// grid = (ceil(max_items / 8), G), block = 256.
template <int NQ>
__global__ void __launch_bounds__(256) k_wide_update_items(WUpdateParams p) {
  __shared__ int first[257];
  const int g = blockIdx.y, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, d = p.d, K = p.K;
  if (group_done(p.st, g, p.t)) return;
  for (int q = tid; q <= K; q += 256) first[q] = p.item_first[(long long)g * (K + 1) + q];
  __syncthreads();
  const int item = blockIdx.x * 8 + warp;
  if (item >= first[K]) return;
  int lo = 0, hi = K - 1;                       // the cluster k with first[k] <= item < first[k + 1]
  while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (first[mid] <= item) lo = mid; else hi = mid - 1; }
  const int k = lo, seg = item - first[k];
  // cluster k's piece of every sub-range list: lane sp holds its length and first position
  int c_sp = 0, pos_sp = 0;
  if (lane < p.nsub) {
    const int *stp = p.starts + ((long long)g * p.nsub + lane) * (K + 1);
    const int s0 = stp[k];
    c_sp = stp[k + 1] - s0;
    pos_sp = (int)wide_sub_begin(p.N, lane, p.nsub) + s0;
  }
  int incl = c_sp;
  for (int off = 1; off < 32; off <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, off); if (lane >= off) incl += v; }
  const int n_k = __shfl_sync(0xffffffffu, incl, 31);
  const int e0 = seg * kItemRows, n_it = min(kItemRows, n_k - e0);
  // entries e0 + lane and e0 + 32 + lane of the cluster's concatenated list
  const int msh = ((p.M & (p.M - 1)) == 0) ? (31 - __clz(p.M)) : -1;
  int row[2] = {0, 0};
  float wv[2] = {0.f, 0.f};
  double wnv[2] = {0.0, 0.0};
  const int *ord = p.order + (long long)g * p.N;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int e = e0 + 32 * h + lane;
    int src = -1;
    for (int sp = 0; sp < p.nsub; ++sp) {
      const int in_sp = __shfl_sync(0xffffffffu, incl, sp), c = __shfl_sync(0xffffffffu, c_sp, sp), ps = __shfl_sync(0xffffffffu, pos_sp, sp);
      if (src < 0 && e < in_sp) src = ps + (e - (in_sp - c));
    }
    if (32 * h + lane < n_it) {
      const int i = ord[src];
      row[h] = i;
      wv[h] = __ldg(p.wt + (long long)g * p.nf_tok + ((msh >= 0) ? (i >> msh) : (i / p.M)));
      wnv[h] = __ldg(p.wn + (long long)g * p.N + i);
    }
  }
  double accA[NQ][4], accB[NQ][4], accW = 0.0;
#pragma unroll
  for (int q = 0; q < NQ; ++q)
#pragma unroll
    for (int j = 0; j < 4; ++j) { accA[q][j] = 0.0; accB[q][j] = 0.0; }
  bool live[NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) live[q] = 4 * lane + 128 * q < d;
  const float *rows_g = p.rows + (long long)g * p.N * d;
  constexpr int kDepth = 8;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    for (int u0 = 0; u0 < 32 && 32 * h + u0 < n_it; u0 += kDepth) {
      float4 x[kDepth][NQ];
#pragma unroll
      for (int u = 0; u < kDepth; ++u) {
        const int i = __shfl_sync(0xffffffffu, row[h], u0 + u);
#pragma unroll
        for (int q = 0; q < NQ; ++q)
          x[u][q] = (32 * h + u0 + u < n_it && live[q]) ? __ldg(reinterpret_cast<const float4 *>(rows_g + (long long)i * d + 4 * lane + 128 * q))
                                                          : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int u = 0; u < kDepth; ++u) {
        const double w_ = (double)__shfl_sync(0xffffffffu, wv[h], u0 + u), wn_ = __shfl_sync(0xffffffffu, wnv[h], u0 + u);
        if (32 * h + u0 + u < n_it) {
#pragma unroll
          for (int q = 0; q < NQ; ++q) {
            const double v[4] = {(double)x[u][q].x, (double)x[u][q].y, (double)x[u][q].z, (double)x[u][q].w};
#pragma unroll
            for (int j = 0; j < 4; ++j) { accA[q][j] = fma(w_, v[j], accA[q][j]); accB[q][j] = fma(wn_, v[j], accB[q][j]); }
          }
          accW += w_;
        }
      }
    }
  }
  double *out = p.part + ((long long)g * p.max_items + item) * (2 * d + 2);
#pragma unroll
  for (int q = 0; q < NQ; ++q)
    if (live[q]) {
      const int e = 4 * lane + 128 * q;
      *reinterpret_cast<double2 *>(out + e) = make_double2(accA[q][0], accA[q][1]);
      *reinterpret_cast<double2 *>(out + e + 2) = make_double2(accA[q][2], accA[q][3]);
      *reinterpret_cast<double2 *>(out + d + e) = make_double2(accB[q][0], accB[q][1]);
      *reinterpret_cast<double2 *>(out + d + e + 2) = make_double2(accB[q][2], accB[q][3]);
    }
  if (lane == 0) { out[2 * d] = accW; out[2 * d + 1] = (double)n_it; }
}

// A cluster's items merged in item order (= ascending rows), then Eq. 7 / Eq. 8.  grid = (K, G), block = 256.
__global__ void __launch_bounds__(256) k_wide_update_items_finish(WUpdateParams p) {
  __shared__ double fin[2 * kMaxD + 2];
  __shared__ double red[256];
  const int k = blockIdx.x, g = blockIdx.y, tid = threadIdx.x;
  if (group_done(p.st, g, p.t)) return;
  const int d = p.d;
  const int i0 = p.item_first[(long long)g * (p.K + 1) + k], i1 = p.item_first[(long long)g * (p.K + 1) + k + 1];
  const double *in = p.part + ((long long)g * p.max_items + i0) * (2 * d + 2);
  for (int v = tid; v < 2 * d + 2; v += 256) {
    double sum = 0.0;
    for (int q = 0; q < i1 - i0; ++q) sum += in[(long long)q * (2 * d + 2) + v];
    fin[v] = sum;
  }
  __syncthreads();
  wide_finish_cluster(p, g, k, fin, red);
}

__device__ __forceinline__ void wide_finish_cluster(const WUpdateParams &p, int g, int k, const double *fin, double *red) {
  const int tid = threadIdx.x, d = p.d;
  // block-wide sums in a fixed tree order
  auto block_sum = [&](double v) -> double {
    red[tid] = v;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) { if (tid < s) red[tid] += red[tid + s]; __syncthreads(); }
    const double r = red[0];
    __syncthreads();
    return r;
  };
  float *s = p.shapes + ((long long)g * p.cb_stride_g + k) * d;
  float *gp = p.gains + (long long)g * p.cb_stride_g + k;
  const double W = fin[2 * d];
  const long long cnt = (long long)fin[2 * d + 1];
  const float g_old_f = *gp;
  const double g_old = (double)g_old_f;
  const int e = tid;   // element handled here (d <= 256)
  const float s_old = (e < d) ? s[e] : 0.0f;
  if (p.mode == 2) {   // KM: centroid = weighted mean; empty cluster keeps its centroid
    const double mu_old2 = block_sum((e < d) ? (double)s_old * (double)s_old : 0.0);
    const double dot_old = block_sum((e < d) ? fin[e] * (double)s_old : 0.0);
    if (tid == 0 && p.term) p.term[((long long)g * p.term_stride + p.t) * p.term_k + k] = 2.0 * dot_old - W * mu_old2;   // sum over the cluster of w (2 x.mu - ||mu||^2)
    if (cnt != 0 && W > 0.0 && e < d) s[e] = (float)(fin[e] / W);
    if (tid == 0 && p.st && cnt == 0) atomicAdd(&p.st[g].n_empty[p.t], 1);
    return;
  }
  const double proj_old = block_sum((e < d) ? fin[e] * (double)s_old : 0.0);
  const double tk = 2.0 * g_old * proj_old - W * g_old * g_old;
  float g_new = g_old_f;
  float s_new = s_old;
  if (cnt != 0 && W > 0.0) {
    if (p.mode == 1) {
      const double bn2 = block_sum((e < d) ? fin[d + e] * fin[d + e] : 0.0);
      const double bn = sqrt(bn2);
      if (bn / W > kDelta && e < d) s_new = (float)(fin[d + e] / bn);
    }
    const double proj = block_sum((e < d) ? fin[e] * (double)s_new : 0.0);
    const double gk = proj / W;
    g_new = (float)(gk > 0.0 ? gk : 0.0);
  }
  if (e < d) s[e] = s_new;
  if (tid == 0) {
    *gp = g_new;
    if (p.mode == 1 && p.term) p.term[((long long)g * p.term_stride + p.t) * p.term_k + k] = tk;
    if (p.gmax) atomicMax(p.gmax + g, __float_as_int(g_new));
    if (p.st) {
      atomicMax(&p.st[g].gmax_bits[p.t + 1], __float_as_int(g_new));
      if (cnt == 0) atomicAdd(&p.st[g].n_empty[p.t], 1);
    }
  }
}

// Alg. 1 l.15-16 after pass t: assignments unchanged -> the group is done.  grid = 1, block = G (<= 1024).
__global__ void k_wide_converged(DevStats *st, int G, int t) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g < G && t > 1 && st[g].done_iter == 0 && st[g].changed[t] == 0) st[g].done_iter = t;
}

// ---------------------------------------------------------------------------------------------------- subtract / decode
struct WSubParams {
  float *rows;            // [G][N][d] residual, updated in place
  long long N;
  int d, K;
  const float *shapes;    // stage slice
  const float *gains;
  long long cb_stride_g;
  const uint8_t *idx;     // [G][N]
  uint8_t *codes;         // code plane of this stage [G][N] (may be idx itself) or nullptr
  __nv_bfloat16 *ahi, *alo;   // operand planes of the NEW residual, or nullptr
  float *rnorm;
};

// r <- fl32(r - fl32(g_k s_k)), element-wise, no contraction (reading c-P).  warp per row; grid = (ceil(N / 8), G).
__global__ void __launch_bounds__(256) k_wide_subtract(WSubParams p) {
  const int g = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long i = (long long)blockIdx.x * 8 + warp;
  if (i >= p.N) return;
  const long long gi = (long long)g * p.N + i;
  const int k = min((int)p.idx[gi], p.K - 1);   // a caller-supplied code >= K must not index past the codebook
  if (p.codes && lane == 0) p.codes[gi] = (uint8_t)k;
  const float gk = p.gains[(long long)g * p.cb_stride_g + k];
  const float *s = p.shapes + ((long long)g * p.cb_stride_g + k) * p.d;
  double n2 = 0.0;
  for (int e0 = lane * 4; e0 < p.d; e0 += 128) {
    float4 r = *reinterpret_cast<float4 *>(p.rows + gi * p.d + e0);
    const float4 sv = *reinterpret_cast<const float4 *>(s + e0);
    r.x = __fsub_rn(r.x, __fmul_rn(gk, sv.x)); r.y = __fsub_rn(r.y, __fmul_rn(gk, sv.y));
    r.z = __fsub_rn(r.z, __fmul_rn(gk, sv.z)); r.w = __fsub_rn(r.w, __fmul_rn(gk, sv.w));
    *reinterpret_cast<float4 *>(p.rows + gi * p.d + e0) = r;
    if (p.ahi) {
      const float x[4] = {r.x, r.y, r.z, r.w};
      uint32_t h[2], l[2];
#pragma unroll
      for (int u = 0; u < 4; u += 2) {
        const __nv_bfloat16 h0 = __float2bfloat16_rn(x[u]), h1 = __float2bfloat16_rn(x[u + 1]);
        const __nv_bfloat16 l0 = __float2bfloat16_rn(__fsub_rn(x[u], __bfloat162float(h0)));
        const __nv_bfloat16 l1 = __float2bfloat16_rn(__fsub_rn(x[u + 1], __bfloat162float(h1)));
        h[u / 2] = (uint32_t)__bfloat16_as_ushort(h0) | ((uint32_t)__bfloat16_as_ushort(h1) << 16);
        l[u / 2] = (uint32_t)__bfloat16_as_ushort(l0) | ((uint32_t)__bfloat16_as_ushort(l1) << 16);
      }
      *reinterpret_cast<uint2 *>(p.ahi + gi * p.d + e0) = make_uint2(h[0], h[1]);
      *reinterpret_cast<uint2 *>(p.alo + gi * p.d + e0) = make_uint2(l[0], l[1]);
      n2 += (double)r.x * r.x + (double)r.y * r.y + (double)r.z * r.z + (double)r.w * r.w;
    }
  }
  if (p.rnorm) {
    for (int off = 16; off; off >>= 1) n2 += __shfl_xor_sync(0xffffffffu, n2, off);
    if (lane == 0) p.rnorm[gi] = (float)sqrt(n2) * 1.000001f;
  }
}

struct WDecParams {
  const uint8_t *codes;   // [S][G][N]
  const float *shapes;    // [G][S][K][d]
  const float *gains;     // [G][S][K]
  int S, K, G, n_stages, d, M;
  long long N;
  void *out;
  int dtype;
  long long stride_g, stride_t;
};

// xhat = ((c0 + c1) + ...) fp32 in stage order, one RN-even cast.  warp per row (the codeword rows are 4 d bytes wide and
// come from L2: S x 256 x d x 4 bytes per group do not fit in shared memory).  grid = (ceil(N / 8), G), block = 256.
__global__ void __launch_bounds__(256) k_wide_decode(WDecParams p) {
  const int g = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long i = (long long)blockIdx.x * 8 + warp;
  if (i >= p.N) return;
  const long long tok = i / p.M;
  const int m = (int)(i - tok * p.M);
  const long long off = (long long)g * p.stride_g + tok * p.stride_t + (long long)m * p.d;
  for (int e0 = lane * 4; e0 < p.d; e0 += 128) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s = 0; s < p.n_stages; ++s) {
      const int k = min((int)p.codes[((long long)s * p.G + g) * p.N + i], p.K - 1);
      const long long cb = ((long long)g * p.S + s) * p.K + k;
      const float gk = __ldg(p.gains + cb);
      const float4 sv = __ldg(reinterpret_cast<const float4 *>(p.shapes + cb * p.d + e0));
      const float4 c = make_float4(__fmul_rn(gk, sv.x), __fmul_rn(gk, sv.y), __fmul_rn(gk, sv.z), __fmul_rn(gk, sv.w));
      if (s == 0) acc = c;
      else { acc.x = __fadd_rn(acc.x, c.x); acc.y = __fadd_rn(acc.y, c.y); acc.z = __fadd_rn(acc.z, c.z); acc.w = __fadd_rn(acc.w, c.w); }
    }
    if (p.dtype == GSRQ_BF16) {
      const __nv_bfloat16 b0 = __float2bfloat16_rn(acc.x), b1 = __float2bfloat16_rn(acc.y), b2 = __float2bfloat16_rn(acc.z), b3 = __float2bfloat16_rn(acc.w);
      *reinterpret_cast<uint2 *>(reinterpret_cast<uint16_t *>(p.out) + off + e0) =
          make_uint2((uint32_t)__bfloat16_as_ushort(b0) | ((uint32_t)__bfloat16_as_ushort(b1) << 16),
                     (uint32_t)__bfloat16_as_ushort(b2) | ((uint32_t)__bfloat16_as_ushort(b3) << 16));
    } else {
      *reinterpret_cast<float4 *>(reinterpret_cast<float *>(p.out) + off + e0) = acc;
    }
  }
}

// Gather kv rows of ALL tokens into compact fp32 rows (the encode's working residual).  warp per row.
__global__ void __launch_bounds__(256) k_wide_gather(RowSrc src, long long N, float *__restrict__ out) {
  const int g = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long i = (long long)blockIdx.x * 8 + warp;
  if (i >= N) return;
  const int d = src.d;
  const long long tok = i / src.M;
  const int m = (int)(i - tok * src.M);
  for (int e0 = lane * 4; e0 < d; e0 += 128) {
    float4 v;
    if (src.dtype == GSRQ_BF16) {
      const uint2 u = *reinterpret_cast<const uint2 *>(reinterpret_cast<const uint16_t *>(src.kv) + (long long)g * src.stride_g + tok * src.stride_t + (long long)m * d + e0);
      v = make_float4(__uint_as_float(u.x << 16), __uint_as_float(u.x & 0xFFFF0000u), __uint_as_float(u.y << 16), __uint_as_float(u.y & 0xFFFF0000u));
    } else {
      v = *reinterpret_cast<const float4 *>(reinterpret_cast<const float *>(src.kv) + (long long)g * src.stride_g + tok * src.stride_t + (long long)m * d + e0);
    }
    *reinterpret_cast<float4 *>(out + ((long long)g * N + i) * d + e0) = v;
  }
}

// ---------------------------------------------------------------------------------------------------- quality metrics
// PAPER.md:202 / :85: per row e2 = ||x - xhat||^2, | ||x|| - ||xhat|| |, cos(x, xhat), ||xhat||^2, ||x||^2 with xhat = the row's prototype
// (KM: the centroid; GSKM: fl32(g_k s_k)); fp64, element order; warp per row, the CTA's 8 rows added in warp order.
// out: [gridDim.x][5] partial sums.  grid = ceil(N / 8), block = 256.
__global__ void __launch_bounds__(256) k_cluster_metrics(const float *__restrict__ x, long long N, int d, const float *__restrict__ shapes,
                                                         const float *__restrict__ gains, const uint16_t *__restrict__ idx, int km,
                                                         int K, double *__restrict__ out) {
  __shared__ double sh[8][5];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long i = (long long)blockIdx.x * 8 + warp;
  double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (i < N) {
    const int k = min((int)idx[i], K - 1);   // caller-supplied labels: clamped, never read past the codebook
    const float gk = km ? 1.0f : gains[k];
    double e2 = 0.0, nx2 = 0.0, np2 = 0.0, dot = 0.0;
    for (int j = lane; j < d; j += 32) {
      const double a = (double)x[i * d + j];
      const double b = (double)(km ? shapes[(long long)k * d + j] : __fmul_rn(gk, shapes[(long long)k * d + j]));
      e2 += (a - b) * (a - b); nx2 += a * a; np2 += b * b; dot += a * b;
    }
    for (int off = 16; off; off >>= 1) {
      e2 += __shfl_xor_sync(0xffffffffu, e2, off); nx2 += __shfl_xor_sync(0xffffffffu, nx2, off);
      np2 += __shfl_xor_sync(0xffffffffu, np2, off); dot += __shfl_xor_sync(0xffffffffu, dot, off);
    }
    const double nx = sqrt(nx2), np = sqrt(np2);
    v[0] = e2; v[1] = fabs(nx - np); v[2] = (nx > 0.0 && np > 0.0) ? dot / (nx * np) : 0.0; v[3] = np2; v[4] = nx2;
  }
  if (lane == 0)
    for (int q = 0; q < 5; ++q) sh[warp][q] = v[q];
  __syncthreads();
  if (threadIdx.x < 5) {
    double s = 0.0;
    for (int w8 = 0; w8 < 8; ++w8) s += sh[w8][threadIdx.x];
    out[(long long)blockIdx.x * 5 + threadIdx.x] = s;
  }
}

// partial sums [n][5] -> res[4] = {MSE, gain error, cosine, shrinkage ratio}; one block of 5 x 32 threads, fixed order
__global__ void __launch_bounds__(160) k_cluster_metrics_finish(const double *__restrict__ part, long long n, long long N, double *__restrict__ res) {
  __shared__ double tot[5];
  const int q = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double s = 0.0;
  for (long long c = lane; c < n; c += 32) s += part[c * 5 + q];
  for (int off = 16; off; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if (lane == 0) tot[q] = s;
  __syncthreads();
  if (threadIdx.x == 0) { res[0] = tot[0] / (double)N; res[1] = tot[1] / (double)N; res[2] = tot[2] / (double)N; res[3] = tot[3] / tot[4]; }
}

}  // namespace wide
}  // namespace gsrq
