// k_fit_tc.cuh -- the whole GSKM Lloyd loop of one residual stage (Alg. 1) as ONE persistent
// kernel: d = 16, K <= 256.  grid = (nx, G): nx CTAs (one per SM) per codebook group, launched cooperatively; every
// CTA owns a contiguous range of the group's 128-row tiles for the whole fit.  Pass t = 0 is Alg. 1 l.2 (gains by
// Eq. 8 under the max-projection assignment, reading c-I), passes t >= 1 are the Lloyd iterations.  Per pass:
//
//   (a) stage   the group's operand images (B_hi, B_lo, B_bias) and fp32 codebook, global -> shared memory;
//   (b) score   tcgen05 filter + fused arg-max over the CTA's tiles, exact fp64 re-score of the ambiguous rows
//               (k_score_tc.cuh; Eq. 5); assignment bytes out, changed-row count;
//   (c) reduce  the CTA's rows, in batches of 1024 staged by one bulk copy: a per-cluster membership bitmap is built
//               with plain byte stores (each thread owns one byte column, so there are no atomics); thread k then
//               walks cluster k's bitmap row and adds the rows it finds to its own fp64 registers
//               A_k = sum w_i r_i, B_k = sum w_i r_i/(||r_i||+eps), W_k = sum w_i, cnt_k (Eq. 6-8 sums, weighted per
//               reading c-W); after the last batch the CTA's partials [K][34] go to global memory;
//   (d) barrier among the nx CTAs of the group (integer arrive counter in global memory);
//   (e) merge   CTA bx owns clusters k = bx, bx + nx, ...: it adds the nx partials in CTA order, applies Eq. 7 / Eq. 8
//               with the safeguards of PAPER.md:178, stores s_k, g_k, the cluster's term of J, and the cluster's rows
//               of the next pass's operand images;
//   (f) barrier; Alg. 1 l.15-16: leave the loop when no assignment changed (t > 1).
//
// Every floating-point sum has a fixed order (bitmap-walk order within a cluster and batch, batch order, CTA order): same
// inputs => same bits; there are no floating-point atomics (integer atomics: counters, max of a bit pattern, the
// barrier).  TMEM, the mbarriers and the constant tile are set up once per fit instead of once per pass, and the
// whole fit is one launch.
#pragma once
#include "k_score_tc.cuh"

namespace gsrq {
namespace tc {

constexpr int kFitBatch = 1024;                 // rows per reduction batch
constexpr int kFitWarps = kThreads / 32;        // 10
constexpr int kFitP = 2 * kD + 2;               // partial record: A[16] | B[16] | W | cnt
// shared memory (offsets from the 1024-byte aligned base).  Phase (c) reuses the (idle) A ring for the staged rows.
constexpr uint32_t kFitSmemOnes = 0;                                         // constant A_1 tile
constexpr uint32_t kFitSmemA = kFitSmemOnes + kPlaneBytes;                   // ring of kStages x 2 planes | rows of a batch
constexpr uint32_t kFitSmemB = kFitSmemA + kStages * 2 * kPlaneBytes;        // 3 operand images
constexpr uint32_t kFitSmemQ = kFitSmemB + 3 * kBImgBytes;                   // deferred exact re-scores
constexpr uint32_t kFitSmemSh = kFitSmemQ + kQCap * 8 + 16;                  // fp32 codebook + gains
constexpr uint32_t kFitSmemBar = kFitSmemSh + kN * kD * 4 + kN * 4;          // mbarriers, TMEM slot
constexpr uint32_t kFitSmemBits = kFitSmemBar + 256;                         // bitmap [256][32] words
constexpr uint32_t kFitSmemCoef = kFitSmemBits + kN * (kFitBatch / 32) * 4;  // [1024] {w_i, w_i/(||r_i||+eps)} fp64
constexpr uint32_t kFitSmemFin = kFitSmemCoef + kFitBatch * 16;              // [20][34] fp64 merged sums of a chunk of clusters
constexpr uint32_t kFitSmemMisc = kFitSmemFin + 2 * kFitWarps * kFitP * 8;   // flags
constexpr uint32_t kFitSmemTotal = kFitSmemMisc + 64 + 1024;                 // + alignment slack
static_assert(kFitBatch * kD * 4 <= kStages * 2 * kPlaneBytes, "the staged rows of a batch reuse the A ring");
static_assert(kFitSmemB % 1024 == 0 && kFitSmemBits % 16 == 0 && kFitSmemCoef % 16 == 0 && kFitSmemTotal <= 227 * 1024, "shared-memory budget / alignment");

struct FitTcParams {
  uint8_t *bimg;           // [G][3][8192] operand images of the codebook scored next (pass 0: written by k_init_ids)
  float *shapes;           // stage slice; codeword k of group g at shapes + (g*cb_stride_g + k)*16
  float *gains;
  long long cb_stride_g;
  const float *rnorm;      // [G][N] fp32 upper bounds of ||r_i||
  const float *rows;       // [G][N][16] fp32 rows
  const __nv_bfloat16 *ahi;  // [G][N][16] bf16 rows (exact when n_planes == 1)
  const double *wn;        // [G][N] w_i / (||r_i|| + eps)
  const float *wt;         // [G][nf_tok] weights of the fit tokens (row i belongs to token i / M)
  long long nf_tok;
  int M;
  uint8_t *idx;            // [G][N] assignment (read as k_old, rewritten every pass)
  long long N;
  int n_tiles, n_planes, K;
  int t_begin, t_end;      // passes [t_begin, t_end]
  int skip_scoring;        // 1: idx is given (step-wise gsrq_update): only (c)-(e) of pass t_begin run
  int lloyd_override;      // -1: pass t updates shapes iff t > 0; 0 / 1: forced (step-wise update)
  DevStats *st;            // [G] or nullptr
  double *term;            // [G][term_stride][256] per-cluster terms of J, or nullptr
  int term_stride;
  double *part;            // [G][nx][256][34] per-CTA partials
  unsigned int *bar;       // [G] arrive counters of the group barrier (zero at launch)
  long long *clk;          // debug: [G][nx][16] cycles per phase (GSRQ_FIT_CLOCKS), or nullptr
};

// Barrier among the CTAs of one group: arrive on an integer counter in global memory, spin until `target` arrivals.
// The CTAs are co-resident (cooperative launch, one per SM).  A bounded spin: a lost CTA ends the wait (and flags the
// fit as failed) instead of hanging the device.
__device__ __forceinline__ void group_barrier(unsigned int *ctr, unsigned int target, DevStats *st) {
  __syncthreads();   // every thread's writes happen-before thread 0's release below (cumulativity)
  if (threadIdx.x == 0) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(ctr), "r"(1u) : "memory");
    unsigned int v = 0;
    long long spins = 0;
    for (;;) {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
      if (v >= target) break;
      if (++spins > (1LL << 26)) { if (st) st->err = GSRQ_ECUDA; break; }
    }
  }
  __syncthreads();
}

__global__ void __launch_bounds__(kThreads, 1)
k_fit_tc(const __grid_constant__ CUtensorMap tm_hi, const __grid_constant__ CUtensorMap tm_lo, FitTcParams p) {
  extern __shared__ uint8_t smem_raw[];
  const int g = blockIdx.y, bx = blockIdx.x, nx = gridDim.x;
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *sgen = smem_raw + (sbase - smem_u32(smem_raw));
  const uint32_t bar0 = sbase + kFitSmemBar;
  auto full_a = [&](int s) { return bar0 + 8u * s; };
  auto empty_a = [&](int s) { return bar0 + 8u * (kStages + s); };
  auto tmem_full = [&](int b) { return bar0 + 8u * (2 * kStages + b); };
  auto tmem_empty = [&](int b) { return bar0 + 8u * (2 * kStages + 2 + b); };
  const uint32_t rows_full = bar0 + 8u * (2 * kStages + 4);
  volatile uint32_t *tmem_slot = reinterpret_cast<volatile uint32_t *>(sgen + kFitSmemBar + 8 * (2 * kStages + 5));
  uint2 *queue = reinterpret_cast<uint2 *>(sgen + kFitSmemQ);
  unsigned int *qcnt = reinterpret_cast<unsigned int *>(sgen + kFitSmemQ + kQCap * 8);
  float *sh_g = reinterpret_cast<float *>(sgen + kFitSmemSh);
  float *ga_g = sh_g + kN * kD;
  uint32_t *bits = reinterpret_cast<uint32_t *>(sgen + kFitSmemBits);
  double2 *coef_s = reinterpret_cast<double2 *>(sgen + kFitSmemCoef);
  double *fin_all = reinterpret_cast<double *>(sgen + kFitSmemFin);
  volatile long long *misc = reinterpret_cast<volatile long long *>(sgen + kFitSmemMisc);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, tid = threadIdx.x;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(full_a(s), 1); mbar_init(empty_a(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tmem_full(b), 1); mbar_init(tmem_empty(b), 4); }
    mbar_init(rows_full, 1);
    fence_barrier_init();
  }
  // constant A_1 tile: columns 0,1,2 = 1.0 (bf16 0x3F80), rest 0
  for (int e = tid; e < kTileM * kD; e += kThreads) {
    const int row = e >> 4, col = e & 15;
    *reinterpret_cast<uint16_t *>(sgen + kFitSmemOnes + sw32_off(row, col)) = (col < 3) ? 0x3F80 : 0;
  }
  fence_proxy_async();
  if (warp == 1) tmem_alloc(smem_u32((const void *)tmem_slot), 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  // this CTA's tiles and rows of group g
  const int tb = (int)((long long)p.n_tiles * bx / nx), te = (int)((long long)p.n_tiles * (bx + 1) / nx);
  const int n_my = te - tb;
  const long long r0 = (long long)tb * kTileM, r1 = min(p.N, (long long)te * kTileM);
  DevStats *stg = p.st ? p.st + g : nullptr;
  const float *shapes_g = p.shapes + (long long)g * p.cb_stride_g * kD;
  const float *gains_g = p.gains + (long long)g * p.cb_stride_g;
  const float rho17 = (p.n_planes == 1 ? 2.0f : 4.5f) * 7.62939453125e-6f;  // rho 2^-17
  const int msh = ((p.M & (p.M - 1)) == 0) ? (31 - __clz(p.M)) : -1;
  const bool rows_bf16 = p.n_planes == 1;
  int tbase = 0;             // tiles this CTA has pushed through the pipeline in earlier passes (ring / accumulator phases)
  unsigned int n_batches = 0;  // reduction batches so far (phase of rows_full)
  unsigned int epoch = 0;      // group barriers passed

  long long clk_last = p.clk ? clock64() : 0;
  auto clk_mark = [&](int phase) {   // debug only (GSRQ_FIT_CLOCKS): cycles spent since the previous mark, by thread 0
    if (p.clk && tid == 0) {
      const long long now = clock64();
      p.clk[((long long)g * nx + bx) * 16 + phase] += now - clk_last;
      clk_last = now;
    }
  };
  for (int t = p.t_begin; t <= p.t_end; ++t) {
    const int mode = (t == 0) ? 1 : 0;
    const int lloyd = (p.lloyd_override >= 0) ? p.lloyd_override : (t > 0 ? 1 : 0);
    // ---------------- (a) operand images and fp32 codebook of the group -> shared memory ----------------
    if (!p.skip_scoring) {
      const uint4 *src = reinterpret_cast<const uint4 *>(p.bimg + (size_t)g * 3 * kBImgBytes);
      uint4 *dst = reinterpret_cast<uint4 *>(sgen + kFitSmemB);
      for (int e = tid; e < (int)(3 * kBImgBytes / 16); e += kThreads) dst[e] = __ldcg(src + e);
      const float4 *s4 = reinterpret_cast<const float4 *>(shapes_g);
      for (int e = tid; e < p.K * (kD / 4); e += kThreads) reinterpret_cast<float4 *>(sh_g)[e] = __ldcg(s4 + e);
      for (int e = tid; e < p.K; e += kThreads) ga_g[e] = __ldcg(gains_g + e);
      if (tid == 0) *qcnt = 0;
      fence_proxy_async();   // generic-proxy writes of the images -> visible to the tensor core's async proxy
    }
    __syncthreads();
    clk_mark(0);

    // ---------------- (b) scoring + arg-max over my tiles ----------------
    if (!p.skip_scoring) {
      if (warp == 0) {
        if (lane == 0) {
          for (int it = 0; it < n_my; ++it) {
            const int gt = tbase + it, st = gt % kStages, ph = (gt / kStages) & 1;
            mbar_wait(empty_a(st), ph ^ 1);
            mbar_expect_tx(full_a(st), p.n_planes * kPlaneBytes);
            tma_load_3d(sbase + kFitSmemA + st * 2 * kPlaneBytes, &tm_hi, 0, (tb + it) * kTileM, g, full_a(st));
            if (p.n_planes == 2)
              tma_load_3d(sbase + kFitSmemA + st * 2 * kPlaneBytes + kPlaneBytes, &tm_lo, 0, (tb + it) * kTileM, g, full_a(st));
          }
        }
      } else if (warp == 1) {
        if (lane == 0) {
          const uint64_t d_bhi = make_desc_sw32(sbase + kFitSmemB), d_blo = make_desc_sw32(sbase + kFitSmemB + kBImgBytes);
          const uint64_t d_bias = make_desc_sw32(sbase + kFitSmemB + 2 * kBImgBytes), d_ones = make_desc_sw32(sbase + kFitSmemOnes);
          for (int it = 0; it < n_my; ++it) {
            const int gt = tbase + it, st = gt % kStages, ph = (gt / kStages) & 1;
            const int buf = gt & 1, bph = (gt >> 1) & 1;
            mbar_wait(tmem_empty(buf), bph ^ 1);
            mbar_wait(full_a(st), ph);
            tc_fence_after();
            const uint32_t d = tmem_base + buf * kN;
            const uint64_t d_ahi = make_desc_sw32(sbase + kFitSmemA + st * 2 * kPlaneBytes);
            mma_f16(d, d_ahi, d_bhi, kIdesc, 0);
            mma_f16(d, d_ahi, d_blo, kIdesc, 1);
            if (p.n_planes == 2) mma_f16(d, make_desc_sw32(sbase + kFitSmemA + st * 2 * kPlaneBytes + kPlaneBytes), d_bhi, kIdesc, 1);
            mma_f16(d, d_ones, d_bias, kIdesc, 1);
            mma_commit(empty_a(st));
            mma_commit(tmem_full(buf));
          }
        }
      } else {
        // Epilogue: warpgroup wg owns accumulator buffer wg, i.e. the tiles whose pipeline index has parity wg.
        const int q = warp & 3;        // TMEM lane quarter this warp may access
        const int wg = (warp - 2) >> 2;
        const float gm = (mode == 0) ? __int_as_float(stg ? __ldcg(&stg->gmax_bits[t]) : 0x7f7fffff) : 1.0f;
        unsigned int n_changed = 0, n_refined = 0;
        for (int it = ((tbase & 1) == wg) ? 0 : 1; it < n_my; it += 2) {
          const int gt = tbase + it, buf = wg, bph = (gt >> 1) & 1;
          const long long row = (long long)(tb + it) * kTileM + q * 32 + lane;
          const long long gr = (long long)g * p.N + row;
          float rn = 0.f;
          uint8_t k_old = 0;
          if (row < p.N) { rn = p.rnorm[gr]; k_old = p.idx[gr]; }   // issued before the wait: latency hidden
          mbar_wait(tmem_full(buf), bph);
          tc_fence_after();
          const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + buf * kN;
          float gmA[16], best, second;
          int gi, ji;
          tile_argmax<false>(taddr, gmA, best, second, gi, ji, nullptr, [&]() {
            tc_fence_before();  // accumulator drained: the MMA warp may overwrite this buffer
            __syncwarp();
            if (lane == 0) mbar_arrive(tmem_empty(buf));
          });
          int k_new = gi * 16 + ji;
          const float E2 = decision_margin(best, rn, ga_g[min(k_new, p.K - 1)], gm, rho17, mode);
          const bool flag = (row < p.N) && (best - second <= E2);
          unsigned int m = __ballot_sync(0xffffffffu, flag);
          n_refined += __popc(m);
          if (m) {  // ambiguous rows: queued, re-scored exactly after the CTA's last tile (a full queue: right here)
            const uint32_t gmask = candidate_groups(gmA, best, E2);
            bool queued = false;
            if (flag) {
              const unsigned int pos = atomicAdd(qcnt, 1u);
              queued = pos < (unsigned int)kQCap;
              if (queued) queue[pos] = make_uint2((uint32_t)row, gmask | ((uint32_t)k_old << 16));
            }
            unsigned int mo = __ballot_sync(0xffffffffu, flag && !queued);
            while (mo) {
              const int l = __ffs(mo) - 1;
              mo &= mo - 1;
              const long long gr_l = (long long)g * p.N + (long long)(tb + it) * kTileM + q * 32 + l;
              const int k = refine_row_warp(p.rows + gr_l * kD, sh_g, ga_g, p.K, mode, lane, __shfl_sync(0xffffffffu, gmask, l));
              if (lane == l) k_new = k;
            }
            if (queued) k_new = -1;  // written by the deferred pass
          }
          if (row < p.N && k_new >= 0) {
            n_changed += (k_old != (uint8_t)k_new);
            p.idx[gr] = (uint8_t)k_new;
          }
        }
        // deferred exact re-scores: entry e is taken by epilogue warp e % 8
        asm volatile("bar.sync 1, 256;" ::: "memory");
        {
          const unsigned int nq = min(*qcnt, (unsigned int)kQCap);
          for (unsigned int e = (unsigned int)(warp - 2); e < nq; e += 8) {
            const uint2 en = queue[e];
            const long long gr_e = (long long)g * p.N + en.x;
            const int k = refine_row_warp(p.rows + gr_e * kD, sh_g, ga_g, p.K, mode, lane, en.y & 0xFFFFu);
            if (lane == 0) {
              n_changed += ((en.y >> 16) != (uint32_t)k);
              p.idx[gr_e] = (uint8_t)k;
            }
          }
        }
        if (stg) {
          for (int off = 16; off; off >>= 1) n_changed += __shfl_xor_sync(0xffffffffu, n_changed, off);
          if (lane == 0 && n_changed) atomicAdd(reinterpret_cast<unsigned long long *>(&stg->changed[t]), (unsigned long long)n_changed);
          if (lane == 0 && n_refined) atomicAdd(reinterpret_cast<unsigned long long *>(&stg->refined), (unsigned long long)n_refined);
        }
      }
      tbase += n_my;
      __syncthreads();
    }
    clk_mark(1);

    // ---------------- (c) reduction over my rows, batches of kFitBatch ----------------
    {
      uint8_t *rows_s = sgen + kFitSmemA;   // the staged rows of the batch reuse the (idle) A ring
      const uint8_t *ig = p.idx + (long long)g * p.N;
      // thread k owns cluster k: its sums live in registers for the whole phase
      double accA[kD], accB[kD], accW = 0.0;
      int cnt = 0;
#pragma unroll
      for (int e = 0; e < kD; ++e) { accA[e] = 0.0; accB[e] = 0.0; }
      // Batch pipeline: the coefficients of batch b + 1 are fetched into registers while batch b is added up; the
      // walk clears the bitmap words it consumes, so the bitmap is clean again when the next batch builds its own.
      constexpr int kCoefPer = (kFitBatch + kThreads - 1) / kThreads;   // 4 rows per thread
      float cw[kCoefPer];
      double cn[kCoefPer];
      uint32_t k8[2];   // the 8 assignment bytes of rows 8 tid .. 8 tid + 7 of the batch
      auto fetch_coef = [&](long long b0, int nb) {
#pragma unroll
        for (int u = 0; u < kCoefPer; ++u) {
          const int e = tid + u * kThreads;
          cw[u] = 0.0f; cn[u] = 0.0;
          if (e < nb) {
            const long long gr_ = b0 + e;
            const long long tk_ = (msh >= 0) ? (gr_ >> msh) : (gr_ / p.M);
            cw[u] = p.wt[(long long)g * p.nf_tok + tk_];
            cn[u] = p.wn[(long long)g * p.N + gr_];
          }
        }
        k8[0] = 0; k8[1] = 0;
        if (8 * tid < nb) {
          const uint8_t *ip = ig + b0 + 8 * tid;
          if (((reinterpret_cast<uintptr_t>(ip) & 7) == 0) && 8 * tid + 8 <= nb) {
            const uint2 v = *reinterpret_cast<const uint2 *>(ip);
            k8[0] = v.x; k8[1] = v.y;
          } else {
#pragma unroll
            for (int j = 0; j < 8; ++j)
              if (8 * tid + j < nb) k8[j >> 2] |= (uint32_t)ip[j] << (8 * (j & 3));
          }
        }
      };
      for (int e = tid; e < kN * (kFitBatch / 32) / 4; e += kThreads) reinterpret_cast<uint4 *>(bits)[e] = make_uint4(0, 0, 0, 0);
      if (r0 < r1) fetch_coef(r0, (int)min((long long)kFitBatch, r1 - r0));
      __syncthreads();
      for (long long b0 = r0; b0 < r1; b0 += kFitBatch) {
        const int nb = (int)min((long long)kFitBatch, r1 - b0);
        const uint32_t row_bytes = rows_bf16 ? 32u : 64u;
        if (tid == 0) {
          mbar_expect_tx(rows_full, (uint32_t)nb * row_bytes);
          const uint8_t *src = rows_bf16 ? reinterpret_cast<const uint8_t *>(p.ahi) + ((long long)g * p.N + b0) * 32
                                         : reinterpret_cast<const uint8_t *>(p.rows) + ((long long)g * p.N + b0) * 64;
          bulk_g2s(smem_u32(rows_s), src, (uint32_t)nb * row_bytes, rows_full);
        }
#pragma unroll
        for (int u = 0; u < kCoefPer; ++u) {   // per-row coefficients {w_i, w_i / (||r_i|| + eps)} of this batch
          const int e = tid + u * kThreads;
          if (e < nb) coef_s[e] = make_double2((double)cw[u], cn[u]);
        }
        clk_mark(11);
        // membership bitmap: thread j owns byte column j (rows 8j..8j+7) of every cluster's 128-byte row: no races
        if (8 * tid < nb) {
          uint8_t *bb = reinterpret_cast<uint8_t *>(bits);
#pragma unroll
          for (int j = 0; j < 8; ++j)
            if (8 * tid + j < nb) bb[(int)((k8[j >> 2] >> (8 * (j & 3))) & 0xFFu) * (kFitBatch / 8) + tid] |= (uint8_t)(1u << j);
        }
        clk_mark(12);
        if (b0 + kFitBatch < r1) fetch_coef(b0 + kFitBatch, (int)min((long long)kFitBatch, r1 - b0 - kFitBatch));   // in flight during the walk
        clk_mark(13);
        __syncthreads();
        clk_mark(7);
        mbar_wait(rows_full, n_batches & 1);
        n_batches++;
        clk_mark(8);
        // thread k walks the non-empty words of cluster k's bitmap row (word j of the walk is (j + k) & 31: conflict-free, and
        // a fixed function of k) and adds the rows it finds: the lanes of a warp advance through their own rows together
        if (tid < p.K) {
          uint32_t sm = 0;
#pragma unroll
          for (int j = 0; j < kFitBatch / 32; ++j) sm |= (bits[tid * (kFitBatch / 32) + ((j + tid) & 31)] != 0u) ? (1u << j) : 0u;
          const int hf = lane & 1;   // odd lanes read the two 16-byte halves of a bf16 row in the other order: spreads the banks
          while (sm) {
            const int wi = ((__ffs(sm) - 1) + tid) & 31;
            sm &= sm - 1;
            uint32_t word = bits[tid * (kFitBatch / 32) + wi];
            bits[tid * (kFitBatch / 32) + wi] = 0u;
            while (word) {
              const int pr = wi * 32 + (__ffs(word) - 1);
              word &= word - 1;
              const double2 cf = coef_s[pr];
              float x[kD];
              if (rows_bf16) {
                const uint4 va = reinterpret_cast<const uint4 *>(rows_s)[pr * 2 + hf], vb = reinterpret_cast<const uint4 *>(rows_s)[pr * 2 + (hf ^ 1)];
                const uint4 v0 = hf ? vb : va, v1 = hf ? va : vb;
                const uint32_t u[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
#pragma unroll
                for (int e = 0; e < 8; ++e) { x[2 * e] = __uint_as_float(u[e] << 16); x[2 * e + 1] = __uint_as_float(u[e] & 0xFFFF0000u); }
              } else {
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4) {
                  const float4 v = reinterpret_cast<const float4 *>(rows_s)[pr * 4 + q4];
                  x[4 * q4] = v.x; x[4 * q4 + 1] = v.y; x[4 * q4 + 2] = v.z; x[4 * q4 + 3] = v.w;
                }
              }
#pragma unroll
              for (int e = 0; e < kD; ++e) {
                const double xd = (double)x[e];
                accA[e] = fma(cf.x, xd, accA[e]);
                accB[e] = fma(cf.y, xd, accB[e]);
              }
              accW += cf.x;
              cnt += 1;
            }
          }
        }
        __syncthreads();
        clk_mark(10);
      }
      // publish this CTA's partials: record k = A[16] | B[16] | W | cnt
      if (tid < kN) {
        double2 *pk = reinterpret_cast<double2 *>(p.part + (((long long)g * nx + bx) * kN + tid) * kFitP);
#pragma unroll
        for (int e = 0; e < kD / 2; ++e) { pk[e] = make_double2(accA[2 * e], accA[2 * e + 1]); pk[kD / 2 + e] = make_double2(accB[2 * e], accB[2 * e + 1]); }
        pk[kD] = make_double2(accW, (double)cnt);
      }
    }
    clk_mark(2);

    // ---------------- (d) every CTA of the group has published its partials ----------------
    ++epoch;
    group_barrier(p.bar + g, epoch * (unsigned int)nx, stg);
    if (tid == 0) misc[0] = (stg && !p.skip_scoring) ? __ldcg(&stg->changed[t]) : 1;
    clk_mark(3);

    // ---------------- (e) merge + Eq. 7 / Eq. 8 for my clusters k = bx, bx + nx, ... ----------------
    // In chunks of 20 clusters: every thread adds up one value of one cluster over the nx partials (CTA order: a fixed
    // order; all loads of a sum in flight together), then one half-warp per cluster applies Eq. 7 / Eq. 8.
    {
      const int ncl = (p.K - bx + nx - 1) / nx;
      const int hw = warp * 2 + (lane >> 4), l16 = lane & 15;
      const unsigned int hmask = 0xFFFFu << (16 * (lane >> 4));
      for (int cl0 = 0; cl0 < ncl; cl0 += 2 * kFitWarps) {
        const int nc = min(2 * kFitWarps, ncl - cl0);
        for (int it = tid; it < nc * kFitP; it += kThreads) {
          const int jj = it / kFitP, v = it - jj * kFitP;
          const double *pp = p.part + ((long long)g * nx * kN + (bx + nx * (cl0 + jj))) * kFitP + v;
          double sum = 0.0;
          for (int c0 = 0; c0 < nx; c0 += 16) {
            double a1[16];
#pragma unroll
            for (int u = 0; u < 16; ++u) a1[u] = (c0 + u < nx) ? __ldcg(pp + (long long)(c0 + u) * kN * kFitP) : 0.0;
#pragma unroll
            for (int u = 0; u < 16; ++u) sum += a1[u];
          }
          fin_all[it] = sum;
        }
        __syncthreads();
        if (hw < nc) {
          const int k = bx + nx * (cl0 + hw);
          const double *f = fin_all + hw * kFitP;
          float *s = p.shapes + ((long long)g * p.cb_stride_g + k) * kD;
          float *gp = p.gains + (long long)g * p.cb_stride_g + k;
          const double W = f[2 * kD], cnt = f[2 * kD + 1];
          const float g_old_f = __ldcg(gp);
          const double g_old = (double)g_old_f;
          float sn[kD];
#pragma unroll
          for (int q4 = 0; q4 < kD / 4; ++q4) {
            const float4 sv = __ldcg(reinterpret_cast<const float4 *>(s) + q4);
            sn[4 * q4] = sv.x; sn[4 * q4 + 1] = sv.y; sn[4 * q4 + 2] = sv.z; sn[4 * q4 + 3] = sv.w;
          }
          __syncwarp(hmask);  // every lane holds the old shape before any lane overwrites it
          double proj_old = 0.0;
#pragma unroll
          for (int jj = 0; jj < kD; ++jj) proj_old += f[jj] * (double)sn[jj];
          const double tk = 2.0 * g_old * proj_old - W * g_old * g_old;  // sum over the cluster of (2 g r.s - g^2) w
          float g_new = g_old_f;
          bool new_shape = false;
          if (cnt != 0.0 && W > 0.0) {
            if (lloyd) {
              double bn2 = 0.0;
#pragma unroll
              for (int jj = 0; jj < kD; ++jj) bn2 = __dadd_rn(bn2, __dmul_rn(f[kD + jj], f[kD + jj]));
              const double bn = sqrt(bn2);
              if (bn / W > kDelta) {  // else: "numerically close to zero": keep the previous shape
                new_shape = true;
                const float mine_new = (float)(f[kD + l16] / bn);
#pragma unroll
                for (int jj = 0; jj < kD; ++jj) sn[jj] = __shfl_sync(hmask, mine_new, jj, 16);
              }
            }
            double proj = 0.0;
#pragma unroll
            for (int jj = 0; jj < kD; ++jj) proj = __dadd_rn(proj, __dmul_rn(f[jj], (double)sn[jj]));
            const double gk = proj / W;
            g_new = (float)(gk > 0.0 ? gk : 0.0);
          }
          float mine = 0.f;
#pragma unroll
          for (int jj = 0; jj < kD; ++jj) if (jj == l16) mine = sn[jj];
          if (new_shape) s[l16] = mine;
          if (p.bimg) write_bimg_elem(p.bimg + (size_t)g * 3 * kBImgBytes, k, l16, g_new, mine, 0, false);
          if (l16 == 0) {
            *gp = g_new;
            if (lloyd && p.term) p.term[((long long)g * p.term_stride + t) * 256 + k] = tk;
            if (stg) {
              atomicMax(&stg->gmax_bits[t + 1], __float_as_int(g_new));
              if (cnt == 0.0) atomicAdd(&stg->n_empty[t], 1);
            }
          }
        }
        __syncthreads();
      }
    }
    clk_mark(4);
    // ---------------- (f) the new codebook is complete; Alg. 1 l.15-16 ----------------
    ++epoch;
    group_barrier(p.bar + g, epoch * (unsigned int)nx, stg);
    clk_mark(5);
    if (lloyd && t > 1 && !p.skip_scoring && misc[0] == 0) {  // assignments unchanged: this was the last iteration
      if (bx == 0 && tid == 0 && stg) stg->done_iter = t;
      break;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, 512);
}

}  // namespace tc
}  // namespace gsrq
