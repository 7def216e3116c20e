// k_update.cuh -- deterministic segmented weighted centroid reduction (sums of Eq. 6-8),
// codeword renormalisation (Eq. 7, Eq. 8, safeguards of PAPER.md:178) and the tensor-core
// operand images of the updated codewords, in ONE "cluster-owner" kernel.
//
// Per cluster k the update needs  cnt_k, W_k = sum w_i, A_k = sum w_i r_i, B_k = sum w_i y_i,
// y_i = r_i/(||r_i||+eps).  A CTA owns kCPC consecutive clusters of one group: it scans the
// group's assignment bytes in passes, compacts the rows of its clusters into an ascending list
// (a stable counting sort: integer work only), stages those rows in shared memory with one
// wave of independent loads, and one warp per cluster adds them up in fp64 in ascending row
// order -- the definition's own order, so A_k, W_k are bit-identical to a sequential fp64 loop
// and B_k differs only by the rounding of w_i/(||r_i||+eps).  A cluster that
// holds more than kBigRows rows of a pass is instead added by all warps, one contiguous chunk each, and the
// chunk partials are merged in chunk order (still a fixed order).  No floating-point atomics, no
// cross-CTA partials: bit-identical run to run.  The same CTA then applies
// Eq. 7 / Eq. 8 to its clusters, stores s_k, g_k, the per-cluster term of J (Eq. 4 summed over
// the cluster), the cluster's rows of the B operand images for the next scoring pass, and
// max g (integer atomicMax on the bit pattern: order-independent).
#pragma once
#include "gsrq_common.cuh"

namespace gsrq {

constexpr int kCPC = 16;            // clusters per CTA = warps per CTA (warp c sums cluster k0 + c)
constexpr int kUpdThreads = 512;
constexpr int kPassRows = 16384;    // rows scanned per pass (32 per thread)
constexpr int kRoundRows = 1024;    // staged rows in shared memory: two buffers of kHalfRows
constexpr int kHalfRows = kRoundRows / 2;

struct UpdParams {
  const float *Rf;        // [G][Nf][D] fp32 rows
  const double2 *coef;    // [G][Nf]   per-row {w_i, w_i/(||r_i||+eps)}
  const uint8_t *idx;     // [G][Nf]
  long long Nf;
  int M, K;
  float *shapes;          // stage slice: shapes + (g*cb_stride_g + k)*D
  float *gains;
  long long cb_stride_g;
  DevStats *st;           // may be nullptr (step-wise gsrq_update)
  double *term;           // [G][term_stride][256] or nullptr
  int term_stride;
  int lloyd;              // 0: gains only (Alg. 1 l.2); 1: shapes + gains
  int t;                  // pass index (slot of changed[], n_empty[], gmax_bits[t+1])
  uint8_t *bimg;          // [G][3][8192] operand images (D == 16 only) or nullptr
};

// byte offset of element (row, col) of a [rows][16] bf16 tile in the SWIZZLE_32B K-major layout
__host__ __device__ __forceinline__ uint32_t sw32_off(int row, int col) {
  return (uint32_t)row * 32u + ((((uint32_t)col >> 3) ^ (((uint32_t)row >> 2) & 1u)) << 4) + ((uint32_t)col & 7u) * 2u;
}
constexpr uint32_t kBImgBytesU = 256 * 16 * 2;

// Write row k of the three operand images (B_hi, B_lo, B_bias) for codeword (gk, s[0..16)):
//   mode 0: c' = fl32(2 fl32(g_k s_kj)), b = fl32(g_k^2);   mode 1 (projection): c' = 2 s_kj, b = 0;
//   dead rows (k >= K) get c' = 0, b = 3e38 so that they can never win the arg-max.
__device__ __forceinline__ void write_bimg_elem(uint8_t *img, int k, int j, float gk, float sj, int mode, bool dead) {
  float c = 0.f;
  if (!dead) c = (mode == 0) ? 2.0f * __fmul_rn(gk, sj) : 2.0f * sj;
  const __nv_bfloat16 hi = __float2bfloat16_rn(c);
  const __nv_bfloat16 lo = __float2bfloat16_rn(__fsub_rn(c, __bfloat162float(hi)));
  *reinterpret_cast<__nv_bfloat16 *>(img + sw32_off(k, j)) = hi;
  *reinterpret_cast<__nv_bfloat16 *>(img + kBImgBytesU + sw32_off(k, j)) = lo;
  const float b = dead ? 3.0e38f : ((mode == 0) ? __fmul_rn(gk, gk) : 0.0f);
  const __nv_bfloat16 b1 = __float2bfloat16_rn(b);
  const float r1 = __fsub_rn(b, __bfloat162float(b1));
  const __nv_bfloat16 b2 = __float2bfloat16_rn(r1);
  const __nv_bfloat16 b3 = __float2bfloat16_rn(__fsub_rn(r1, __bfloat162float(b2)));
  __nv_bfloat16 v = __float2bfloat16_rn(0.f);
  if (j == 0) v = __hneg(b1);
  if (j == 1) v = __hneg(b2);
  if (j == 2) v = __hneg(b3);
  *reinterpret_cast<__nv_bfloat16 *>(img + 2 * kBImgBytesU + sw32_off(k, j)) = v;
}

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}

// 4 assignment bytes of rows [r, r+4) of one group; rows >= Nf read as `miss`.
__device__ __forceinline__ uint32_t load_idx_word(const uint8_t *ig, long long r, long long Nf, bool aligned, uint32_t miss) {
  if (aligned && r + 4 <= Nf) return *reinterpret_cast<const uint32_t *>(ig + r);
  uint32_t w = 0;
#pragma unroll
  for (int b = 0; b < 4; ++b) {
    const uint32_t v = (r + b < Nf) ? (uint32_t)ig[r + b] : miss;
    w |= v << (8 * b);
  }
  return w;
}

constexpr int kBigRows = 256;  // a cluster with more rows than this in one pass is added by all warps together

// Rows [x0, x1) of the staged round (positions in the pass's list; the round starts at `lo`) added in list order by
// one warp into a partial of P = 2D + 2 values at `out` (shared memory): [A | B | W | unused].  Cold path of
// k_update, used for clusters that hold hundreds of rows of a pass (heavy-tailed tensors).
template <int D>
__device__ __noinline__ void upd_add_chunk(const float *xbuf_r, const double *coef_r, int x0, int x1, int lo, int lane, double *out) {
  constexpr int Q = (2 * D + 31) / 32;
  double sp[Q], Wp = 0.0;
  int isB[Q], col[Q];
  bool live[Q];
#pragma unroll
  for (int q = 0; q < Q; ++q) {
    const int el = lane + 32 * q;
    sp[q] = 0.0; live[q] = el < 2 * D; isB[q] = (el >= D) ? 1 : 0; col[q] = el % D;
  }
  int pos = x0;
  for (; pos + 4 <= x1; pos += 4) {
    double cf[4][Q];
    float xv[4][Q];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int e = pos + u - lo;
#pragma unroll
      for (int q = 0; q < Q; ++q) {
        cf[u][q] = live[q] ? coef_r[2 * e + isB[q]] : 0.0;
        xv[u][q] = live[q] ? xbuf_r[e * D + col[q]] : 0.0f;
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      Wp += cf[u][0];
#pragma unroll
      for (int q = 0; q < Q; ++q) sp[q] += cf[u][q] * (double)xv[u][q];
    }
  }
  for (; pos < x1; ++pos) {
    const int e = pos - lo;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const double cf = live[q] ? coef_r[2 * e + isB[q]] : 0.0;
      if (q == 0) Wp += cf;
      sp[q] += cf * (double)(live[q] ? xbuf_r[e * D + col[q]] : 0.0f);
    }
  }
#pragma unroll
  for (int q = 0; q < Q; ++q)
    if (live[q]) out[lane + 32 * q] = sp[q];
  if (lane == 0) out[2 * D] = Wp;
}

template <int D>
constexpr size_t upd_smem_bytes() {
  constexpr int P = 2 * D + 2;
  return sizeof(double) * (2 * kRoundRows + kCPC * P) + sizeof(float) * (kRoundRows * D) +
         sizeof(int) * (kCPC + 4) + sizeof(uint16_t) * (kPassRows + kCPC * kUpdThreads) + kPassRows +
         sizeof(double) * (kUpdThreads / 32) * P + sizeof(int) * (kCPC + 4);
}

// grid = (ceil(K / kCPC), G), block = kUpdThreads, dynamic smem = upd_smem_bytes<D>().
template <int D>
__global__ void __launch_bounds__(kUpdThreads, 1) k_update(UpdParams p) {
  extern __shared__ __align__(16) uint8_t upd_sm[];
  constexpr int P = 2 * D + 2;
  constexpr int Q = (2 * D + 31) / 32;
  constexpr int LPR = D / 4;
  static_assert(kCPC * 32 == kUpdThreads && kPassRows == 32 * kUpdThreads, "thread mapping");
  double *coef = reinterpret_cast<double *>(upd_sm);        // [kRoundRows][2]  { w_i, w_i / (||r_i|| + eps) }
  double *fin = coef + 2 * kRoundRows;                      // [kCPC][P]
  float *xbuf = reinterpret_cast<float *>(fin + kCPC * P);  // [kRoundRows][D]
  int *ctot = reinterpret_cast<int *>(xbuf + kRoundRows * D);  // [kCPC] (+4 pad)
  uint16_t *list = reinterpret_cast<uint16_t *>(ctot + kCPC + 4);  // [kPassRows] rows of the pass, by (cluster, row)
  uint16_t *cntb = list + kPassRows;                        // [kCPC][kUpdThreads] per-thread counts -> prefixes
  uint8_t *idxb = reinterpret_cast<uint8_t *>(cntb + kCPC * kUpdThreads);  // [kPassRows] assignment bytes of the pass
  double *part = reinterpret_cast<double *>(idxb + kPassRows);  // [warps][P] chunk partials of a big cluster's segment
  int *cb_s = reinterpret_cast<int *>(part + (kUpdThreads / 32) * P);  // [kCPC + 1] list offsets of the clusters; [kCPC + 1]: mask of big clusters

  const int g = blockIdx.y, k0 = blockIdx.x * kCPC;
  if (group_done(p.st, g, p.t)) return;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint8_t *ig = p.idx + (long long)g * p.Nf;
  const bool aligned = (reinterpret_cast<uintptr_t>(ig) & 3) == 0;
  const bool aligned16 = (reinterpret_cast<uintptr_t>(ig) & 15) == 0;
  const uint32_t pat = (uint32_t)(k0 & 0xF0) * 0x01010101u;
  const uint32_t miss = (uint32_t)((k0 ^ 0x80) & 0xFF);  // a byte outside [k0, k0 + 16)
  const float *rows = p.Rf + (long long)g * p.Nf * D;
  const double2 *cf_g = p.coef + (long long)g * p.Nf;

  double s[Q];  // warp c, lane e: element e (+32q) of [A | B] of cluster k0 + c
  int isB[Q], col[Q];
  bool live[Q];
#pragma unroll
  for (int q = 0; q < Q; ++q) {
    const int el = lane + 32 * q;
    s[q] = 0.0; live[q] = el < 2 * D; isB[q] = (el >= D) ? 1 : 0; col[q] = el % D;
  }
  double Wk = 0.0;
  long long cntk = 0;
  for (long long pb = 0; pb < p.Nf; pb += kPassRows) {
    // ---- walk 1: my 32 assignment bytes -> hit mask, per-(cluster, thread) counts ----
    uint32_t m = 0;
    {
      // the warp stages its 1024 bytes with coalesced 16-byte loads, then each thread takes its 32 rows
      const long long wb = pb + 1024 * warp;
      uint4 *stage = reinterpret_cast<uint4 *>(idxb + 1024 * warp);
      if (aligned16 && wb + 1024 <= p.Nf) {
        const uint4 *src = reinterpret_cast<const uint4 *>(ig + wb);
        const uint4 v0 = __ldg(src + lane), v1 = __ldg(src + 32 + lane);
        stage[lane] = v0;
        stage[32 + lane] = v1;
      } else {
        const long long r0 = wb + 32 * lane;
#pragma unroll
        for (int wi = 0; wi < 8; ++wi)
          reinterpret_cast<uint32_t *>(idxb)[8 * tid + wi] =
              (r0 + 4 * wi < p.Nf) ? load_idx_word(ig, r0 + 4 * wi, p.Nf, aligned, miss) : miss * 0x01010101u;
      }
      __syncwarp();
      const uint4 a0 = stage[2 * lane], a1 = stage[2 * lane + 1];
      const uint32_t w[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
#pragma unroll
      for (int wi = 0; wi < 8; ++wi) {
        uint32_t h = __vcmpeq4(w[wi] & 0xF0F0F0F0u, pat) & 0x08040201u;  // bits 0, 9, 18, 27 <- bytes 0..3 hit
        h = (h | (h >> 8) | (h >> 16) | (h >> 24)) & 0xFu;
        m |= h << (4 * wi);
      }
    }
#pragma unroll
    for (int c = 0; c < kCPC; ++c) cntb[c * kUpdThreads + tid] = 0;
    for (uint32_t mm = m; mm; mm &= mm - 1) {
      const int r = __ffs(mm) - 1;
      const int c = idxb[32 * tid + r] & (kCPC - 1);
      cntb[c * kUpdThreads + tid] += 1;
    }
    __syncthreads();
    // ---- warp c: exclusive prefix of cluster c's counts over the 512 threads (integers) ----
    {
      uint16_t *row = cntb + warp * kUpdThreads + 16 * lane;
      uint4 v0 = reinterpret_cast<uint4 *>(row)[0], v1 = reinterpret_cast<uint4 *>(row)[1];
      uint32_t u[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
      int run = 0;
#pragma unroll
      for (int i = 0; i < 8; ++i) {  // two 16-bit counts per word -> their exclusive prefixes
        const int a = (int)(u[i] & 0xFFFFu), b = (int)(u[i] >> 16);
        u[i] = (uint32_t)run | ((uint32_t)(run + a) << 16);
        run += a + b;
      }
      int incl = run;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += v;
      }
      const uint32_t base2 = (uint32_t)(incl - run) * 0x00010001u;
#pragma unroll
      for (int i = 0; i < 8; ++i) u[i] += base2;
      reinterpret_cast<uint4 *>(row)[0] = make_uint4(u[0], u[1], u[2], u[3]);
      reinterpret_cast<uint4 *>(row)[1] = make_uint4(u[4], u[5], u[6], u[7]);
      if (lane == 31) ctot[warp] = incl;
    }
    __syncthreads();
    // ---- walk 2: stable scatter of my hits, ordered by (cluster, row) ----
    int cbase[kCPC + 1];
    cbase[0] = 0;
#pragma unroll
    for (int c = 0; c < kCPC; ++c) cbase[c + 1] = cbase[c] + ctot[c];
    const int total = cbase[kCPC];
    if (tid == 0) {
      int bm = 0;
#pragma unroll
      for (int c = 0; c < kCPC; ++c) { cb_s[c] = cbase[c]; bm |= (cbase[c + 1] - cbase[c] > kBigRows) ? (1 << c) : 0; }
      cb_s[kCPC] = cbase[kCPC];
      cb_s[kCPC + 1] = bm;
    }
    for (uint32_t mm = m; mm; mm &= mm - 1) {
      const int r = __ffs(mm) - 1;
      const int c = idxb[32 * tid + r] & (kCPC - 1);
      int base = 0;
#pragma unroll
      for (int c2 = 0; c2 < kCPC; ++c2) base = (c2 == c) ? cbase[c2] : base;
      const int pos = base + (int)cntb[c * kUpdThreads + tid];
      cntb[c * kUpdThreads + tid] += 1;
      list[pos] = (uint16_t)(32 * tid + r);
    }
    int seg0 = 0, seg1 = 0;
#pragma unroll
    for (int c2 = 0; c2 < kCPC; ++c2)
      if (c2 == warp) { seg0 = cbase[c2]; seg1 = cbase[c2 + 1]; }
    __syncthreads();
    // Rounds of kHalfRows staged rows, double-buffered: the asynchronous copies of round r + 1 (rows and their
    // coefficient pairs, 16 bytes each, global -> shared) are in flight while round r is added up.
    auto issue = [&](int lo_r, int buf) {
      const int n_r = min(kHalfRows, total - lo_r);
      const int q = tid % LPR;
      float *xb = xbuf + buf * kHalfRows * D;
      double *cb = coef + buf * kHalfRows * 2;
#pragma unroll
      for (int u = 0; u < kHalfRows * LPR / kUpdThreads; ++u) {
        const int e = (tid + u * kUpdThreads) / LPR;
        if (e < n_r) {
          const long long row = pb + list[lo_r + e];
          cp_async16(xb + e * D + 4 * q, rows + row * D + 4 * q);
          if (q == 0) cp_async16(cb + 2 * e, cf_g + row);
        }
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
    };
    if (total > 0) issue(0, 0);
    for (int lo = 0, rd = 0; lo < total; lo += kHalfRows, ++rd) {
      const int n = min(kHalfRows, total - lo);
      if (lo + kHalfRows < total) {
        issue(lo + kHalfRows, (rd + 1) & 1);
        asm volatile("cp.async.wait_group 1;" ::: "memory");
      } else {
        asm volatile("cp.async.wait_group 0;" ::: "memory");
      }
      __syncthreads();
      const float *xbuf_r = xbuf + (rd & 1) * kHalfRows * D;
      const double *coef_r = coef + (rd & 1) * kHalfRows * 2;
      // ---- warp c adds cluster c's rows of this round in list (= ascending row) order ----
      const int bigmask = cb_s[kCPC + 1];  // uniform; zero unless a cluster holds > kBigRows rows of this pass
      const int a = max(seg0, lo), b = ((bigmask >> warp) & 1) ? a : min(seg1, lo + n);
      int pos = a;
      for (; pos + 4 <= b; pos += 4) {  // loads of 4 rows in flight; the adds stay in list order
        double cf[4][Q];
        float xv[4][Q];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int e = pos + u - lo;
#pragma unroll
          for (int q = 0; q < Q; ++q) {
            cf[u][q] = live[q] ? coef_r[2 * e + isB[q]] : 0.0;
            xv[u][q] = live[q] ? xbuf_r[e * D + col[q]] : 0.0f;
          }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          Wk += cf[u][0];  // lane 0 is an A lane: its coefficient is w_i
#pragma unroll
          for (int q = 0; q < Q; ++q) s[q] += cf[u][q] * (double)xv[u][q];
        }
      }
      for (; pos < b; ++pos) {
        const int e = pos - lo;
#pragma unroll
        for (int q = 0; q < Q; ++q) {
          const double cf = live[q] ? coef_r[2 * e + isB[q]] : 0.0;
          if (q == 0) Wk += cf;
          s[q] += cf * (double)(live[q] ? xbuf_r[e * D + col[q]] : 0.0f);
        }
      }
      if (a < b) cntk += b - a;
      __syncthreads();
      // ---- big clusters: the segment is split into one contiguous chunk per warp, added concurrently, and the chunk
      //      partials are merged by the owner warp in warp (= list) order ----
      for (int bmk = bigmask; bmk; bmk &= bmk - 1) {
        const int c = __ffs(bmk) - 1;
        const int ca = max(cb_s[c], lo), cb = min(cb_s[c + 1], lo + n);
        if (ca >= cb) continue;
        const int chunk = (cb - ca + kUpdThreads / 32 - 1) / (kUpdThreads / 32);
        const int x0 = min(ca + warp * chunk, cb), x1 = min(x0 + chunk, cb);
        upd_add_chunk<D>(xbuf_r, coef_r, x0, x1, lo, lane, part + warp * P);
        __syncthreads();
        if (warp == c) {
          double pv[kUpdThreads / 32][Q], pw[kUpdThreads / 32];  // fetch first, then add in warp order
#pragma unroll
          for (int wq = 0; wq < kUpdThreads / 32; ++wq) {
#pragma unroll
            for (int q = 0; q < Q; ++q) pv[wq][q] = live[q] ? part[wq * P + lane + 32 * q] : 0.0;
            pw[wq] = part[wq * P + 2 * D];
          }
#pragma unroll
          for (int wq = 0; wq < kUpdThreads / 32; ++wq) {
#pragma unroll
            for (int q = 0; q < Q; ++q) s[q] += pv[wq][q];
            Wk += pw[wq];
          }
          cntk += cb - ca;
        }
        __syncthreads();
      }
    }
  }
  {
    double *out = fin + warp * P;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int el = lane + 32 * q;
      if (el < 2 * D) out[el] = s[q];
    }
    if (lane == 0) { out[2 * D] = Wk; out[2 * D + 1] = (double)cntk; }
  }
  __syncwarp();
  // ---- Eq. 7 / Eq. 8 for my clusters: warp c, lane j (every lane evaluates the scalar chain) ----
  if (warp < kCPC && k0 + warp < p.K) {
    const int k = k0 + warp;
    const double *f = fin + warp * P;
    float *s = p.shapes + ((long long)g * p.cb_stride_g + k) * D;
    float *gp = p.gains + (long long)g * p.cb_stride_g + k;
    const double W = f[2 * D], cnt = f[2 * D + 1];
    const float g_old_f = *gp;
    const double g_old = (double)g_old_f;
    float sn[D];
#pragma unroll
    for (int j = 0; j < D; ++j) sn[j] = s[j];
    __syncwarp();  // every lane holds the old shape before any lane overwrites it
    double proj_old = 0.0;
#pragma unroll
    for (int j = 0; j < D; ++j) proj_old += f[j] * (double)sn[j];
    const double tk = 2.0 * g_old * proj_old - W * g_old * g_old;  // sum over the cluster of (2 g r.s - g^2) w
    float g_new = g_old_f;
    bool new_shape = false;
    if (cnt != 0.0 && W > 0.0) {
      if (p.lloyd) {
        double bn2 = 0.0;
#pragma unroll
        for (int j = 0; j < D; ++j) bn2 = __dadd_rn(bn2, __dmul_rn(f[D + j], f[D + j]));
        const double bn = sqrt(bn2);
        if (bn / W > kDelta) {
          new_shape = true;
          float *sx = reinterpret_cast<float *>(xbuf) + warp * D;  // xbuf is free now: exchange the new shape
          if (lane < D) sx[lane] = (float)(f[D + lane] / bn);
          __syncwarp();
#pragma unroll
          for (int j = 0; j < D; ++j) sn[j] = sx[j];
        }
      }
      double proj = 0.0;
#pragma unroll
      for (int j = 0; j < D; ++j) proj = __dadd_rn(proj, __dmul_rn(f[j], (double)sn[j]));
      const double gk = proj / W;
      g_new = (float)(gk > 0.0 ? gk : 0.0);
    }
    float mine = 0.f;
#pragma unroll
    for (int j = 0; j < D; ++j) if (j == lane) mine = sn[j];
    if (lane < D && new_shape) s[lane] = mine;
    if (D == 16 && p.bimg && lane < 16)
      write_bimg_elem(p.bimg + (size_t)g * 3 * kBImgBytesU, k, lane, g_new, mine, 0, false);
    if (lane == 0) {
      *gp = g_new;
      if (p.lloyd && p.term) p.term[((long long)g * p.term_stride + p.t) * 256 + k] = tk;
      if (p.st) {
        atomicMax(&p.st[g].gmax_bits[p.t + 1], __float_as_int(g_new));
        if (cnt == 0.0) atomicAdd(&p.st[g].n_empty[p.t], 1);
      }
    }
  }
  // Alg. 1 l.15-16: assignments unchanged -> this was the last iteration of the group
  if (p.st && p.lloyd && p.t > 1 && blockIdx.x == 0 && tid == 0 && p.st[g].changed[p.t] == 0) p.st[g].done_iter = p.t;
}

// Per-group wrap-up of a fit: iters_run, Etot = sum of the energy partials (fixed order) and
// J_t = Etot - sum_k term_t[k] (Eq. 4 summed over rows; k in ascending order).  grid = G, block = 160.
__global__ void __launch_bounds__(160) k_finish(DevStats *__restrict__ st, const double *__restrict__ term, int term_stride,
                                                int K, const double *__restrict__ epart, int n_epart, int iters, int term_k = 256) {
  __shared__ double etot;
  const int g = blockIdx.x, t = threadIdx.x;
  if (t == 0) {
    double e = 0.0;
    for (int c = 0; c < n_epart; ++c) e += epart[(long long)g * n_epart + c];
    etot = e;
    st[g].iters_run = st[g].done_iter ? st[g].done_iter : iters;
  }
  __syncthreads();
  const int n = st[g].done_iter ? st[g].done_iter : iters;
  if (t >= 1 && t <= n) {
    const double *tm = term + ((long long)g * term_stride + t) * term_k;
    double sum = 0.0;
    for (int k = 0; k < K; ++k) sum += tm[k];
    st[g].J[t] = etot - sum;
  }
}

}  // namespace gsrq
