// k_fit_tc.cuh -- the whole GSKM Lloyd loop of one residual stage (Alg. 1) as ONE persistent
// kernel: d = 16, K <= 256.  grid = (nx, G): nx CTAs (one per SM) per codebook group, launched cooperatively; every
// CTA owns a contiguous range of the group's 128-row tiles for the whole fit.  Pass t = 0 is Alg. 1 l.2 (gains by
// Eq. 8 under the max-projection assignment, reading c-I), passes t >= 1 are the Lloyd iterations.  Per pass:
//
//   (a) stage   the group's operand images (B_hi, B_lo, B_bias) and fp32 codebook, global -> shared memory;
//   (b) score   tcgen05 filter + fused arg-max over the CTA's tiles, exact fp64 re-score of the ambiguous rows
//               (k_score_tc.cuh; Eq. 5); assignment bytes out, changed-row count;
//   (c) reduce  the CTA keeps the sums of its own rows per cluster, A_k = sum w_i r_i, B_k = sum w_i r_i/(||r_i||+eps),
//               W_k = sum w_i, cnt_k (Eq. 6-8 sums, weighted per reading c-W), in shared memory as fp64 for the whole
//               fit.  The first pass adds every row; later passes are INCREMENTAL: the scoring epilogue appends the
//               rows whose assignment changed (a few per cent of the rows after the first iterations) to per-warp
//               lists, and the reduce phase subtracts such a row from its old cluster and adds it to its new one.
//               Cluster k belongs to reduce warp k % 8, which walks the lists in a fixed order (warp segment, tile,
//               row), 32 lanes = the 16 elements of A_k and of B_k; the CTA's sums [K][34] then go to global memory;
//   (d) barrier among the nx CTAs of the group (integer arrive counter in global memory);
//   (e) merge   CTA bx owns clusters k = bx, bx + nx, ...: it adds the nx partials in CTA order, applies Eq. 7 / Eq. 8
//               with the safeguards of PAPER.md:178, stores s_k, g_k, the cluster's term of J, and the cluster's rows
//               of the next pass's operand images;
//   (f) barrier; Alg. 1 l.15-16: leave the loop when no assignment changed (t > 1).
//
// Every floating-point sum has a fixed order (list order within a cluster, pass order, CTA order): same
// inputs => same bits; there are no floating-point atomics (integer atomics: counters, max of a bit pattern, the
// barrier).  TMEM, the mbarriers and the constant tile are set up once per fit instead of once per pass, and the
// whole fit is one launch.
#pragma once
#include "k_score_tc.cuh"

namespace gsrq {
namespace tc {

constexpr int kFitWarps = kThreads / 32;        // 10
constexpr int kFitP = 2 * kD + 2;               // partial record: A[16] | B[16] | W | cnt
// shared memory (offsets from the 1024-byte aligned base).  Phase (c) reuses the (idle) A ring for the staged rows.
constexpr uint32_t kFitSmemOnes = 0;                                         // constant A_1 tile
constexpr uint32_t kFitSmemA = kFitSmemOnes + kPlaneBytes;                   // ring of kStages x 2 planes | staging of the reduce warps
constexpr uint32_t kFitSmemB = kFitSmemA + kStages * 2 * kPlaneBytes;        // 3 operand images
constexpr uint32_t kFitSmemQ = kFitSmemB + 3 * kBImgBytes;                   // deferred exact re-scores
constexpr uint32_t kFitSmemSh = kFitSmemQ + kQCap * 8 + 16;                  // fp32 codebook + gains
constexpr uint32_t kFitSmemBar = kFitSmemSh + kN * kD * 4 + kN * 4;          // mbarriers, TMEM slot
constexpr uint32_t kFitSmemAcc = kFitSmemBar + 256;                          // [256][34] fp64: this CTA's sums per cluster (kept over the passes)
constexpr uint32_t kFitSmemFin = kFitSmemAcc + kN * kFitP * 8;               // [20][34] fp64 merged sums of a chunk of clusters
constexpr uint32_t kFitSmemMisc = kFitSmemFin + 2 * kFitWarps * kFitP * 8;   // flags, list lengths
constexpr uint32_t kFitSmemTotal = kFitSmemMisc + 64 + 1024;                 // + alignment slack
constexpr int kFitRedWarps = 8;                                              // reduce warps (= the epilogue warps); cluster k belongs to warp k % 8
constexpr uint32_t kFitStageBytes = 32768 + 4096 + 16384;                    // staging buffer of the reduce phase: 256 x {row fp64, {w, w/(||r||+eps)}} + bitmaps [256][16] words
static_assert(2 * kFitStageBytes <= kFitSmemBar - kFitSmemA, "the two staging buffers of the reduce phase are laid over the scoring-only buffers (A ring, operand images, queue, fp32 codebook)");
static_assert(kFitSmemB % 1024 == 0 && kFitSmemAcc % 16 == 0 && kFitSmemTotal <= 227 * 1024, "shared-memory budget / alignment");

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
  uint2 *chg;              // [G][chg_stride_g] change lists: {row - r0, k_old | k_new << 8 | pending << 17}
  long long chg_stride_g;  // >= 128 n_tiles + 512 nx
  double *part;            // [G][nx][256][34] per-CTA partials
  unsigned int *bar;       // [G] arrive counters of the group barrier (zero at launch)
  long long *clk;          // debug: [G][nx][16] cycles per phase (GSRQ_FIT_CLOCKS), or nullptr
};

// The group's "a barrier wait timed out" flag, read from global memory (never from a stale cache line).
__device__ __forceinline__ bool fit_lost(const DevStats *st) {
  int e = 0;
  if (st) asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(e) : "l"(&st->err) : "memory");
  return e == GSRQ_ECUDA;
}

// Barrier among the CTAs of one group: arrive on an integer counter in global memory, spin until `target` arrivals.
// The CTAs are co-resident (cooperative launch, one per SM).  A bounded spin: a lost CTA ends the wait (and flags the
// fit as failed) instead of hanging the device.  Once the flag is up, the group's other CTAs stop waiting as well (they poll it
// every 4096 spins) and every CTA leaves the pass loop at its next check without touching the codebook again: the caller sees
// GSRQ_ECUDA through `stats` or gsrq_fit_status, never a silently half-updated codebook reported as GSRQ_OK.
__device__ __forceinline__ void group_barrier(unsigned int *ctr, unsigned int target, DevStats *st) {
  __syncthreads();   // every thread's writes happen-before thread 0's release below (cumulativity)
  if (threadIdx.x == 0) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(ctr), "r"(1u) : "memory");
    unsigned int v = 0;
    long long spins = 0;
    for (;;) {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
      if (v >= target) break;
      if (++spins > (1LL << 26)) { if (st) st->err = GSRQ_ECUDA; __threadfence(); break; }
      if ((spins & 4095) == 0 && fit_lost(st)) break;
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
  volatile uint32_t *tmem_slot = reinterpret_cast<volatile uint32_t *>(sgen + kFitSmemBar + 8 * (2 * kStages + 5));
  uint2 *queue = reinterpret_cast<uint2 *>(sgen + kFitSmemQ);
  unsigned int *qcnt = reinterpret_cast<unsigned int *>(sgen + kFitSmemQ + kQCap * 8);
  float *sh_g = reinterpret_cast<float *>(sgen + kFitSmemSh);
  float *ga_g = sh_g + kN * kD;
  double *acc_s = reinterpret_cast<double *>(sgen + kFitSmemAcc);
  double *fin_all = reinterpret_cast<double *>(sgen + kFitSmemFin);
  volatile long long *misc = reinterpret_cast<volatile long long *>(sgen + kFitSmemMisc);
  volatile unsigned int *lcnt = reinterpret_cast<volatile unsigned int *>(sgen + kFitSmemMisc + 16);   // [8] entries in each warp's change list
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, tid = threadIdx.x;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(full_a(s), 1); mbar_init(empty_a(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tmem_full(b), 1); mbar_init(tmem_empty(b), 4); }
    fence_barrier_init();
  }
  // constant A_1 tile: columns 0,1,2 = 1.0 (bf16 0x3F80), rest 0
  for (int e = tid; e < kTileM * kD; e += kThreads) {
    const int row = e >> 4, col = e & 15;
    *reinterpret_cast<uint16_t *>(sgen + kFitSmemOnes + sw32_off(row, col)) = (col < 3) ? 0x3F80 : 0;
  }
  for (int e = tid; e < kN * kFitP; e += kThreads) acc_s[e] = 0.0;
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
  // change lists: the CTA's region starts at entry 128 tb + 512 bx of the group's buffer, one segment per epilogue warp
  const long long cap_w = (long long)(n_my / 2 + 2) * 32;
  uint2 *chg_cta = p.chg + (long long)g * p.chg_stride_g + (long long)tb * kTileM + (long long)bx * 512;
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
    const bool first = (t == p.t_begin);   // the pass that adds every row; later passes move the changed rows only
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
        unsigned int n_changed = 0, n_refined = 0, lc = 0;
        uint2 *seg = chg_cta + (long long)(warp - 2) * cap_w;
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
          if (!first) {  // rows that (may) have moved: appended in row order; a queued row's new cluster is read back from idx later
            const bool ch = (row < p.N) && (k_new < 0 || (uint8_t)k_new != k_old);
            const unsigned int cm = __ballot_sync(0xffffffffu, ch);
            if (ch) seg[lc + __popc(cm & ((1u << lane) - 1u))] =
                make_uint2((uint32_t)(row - r0), (uint32_t)k_old | ((uint32_t)(k_new < 0 ? 0 : k_new) << 8) | (k_new < 0 ? (1u << 17) : 0u));
            lc += __popc(cm);
          }
        }
        if (lane == 0) lcnt[warp - 2] = lc;
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

    // ---------------- (c) this CTA's sums per cluster: add every row (first pass) or move the changed rows ----------------
    // Operations come in batches of 256 list entries, one per thread of warps 2-9.  Fetch (two batches / one batch ahead,
    // into registers): the entry, then its row, weights and -- first pass / queued rows -- its cluster.  Park (staging
    // buffer b & 1, laid over the scoring-only shared memory): the row widened to fp64 (the fp32 -> fp64 conversion runs
    // at 1/8 rate, so it is done once per entry here, not once per use), {w_i, w_i/(||r_i||+eps)}, and one bit per
    // operation in the bitmap row of the cluster it leaves / joins (integer atomicOr: order-free).  Walk: thread k owns
    // cluster k; it loads the cluster's 34 sums into registers, visits the set bits of its bitmap row in order
    // (leaving rows, then joining rows; entry order within each) and stores the sums back after the last batch.
    if (warp >= 2) {
      const int j = tid - 64;    // entry of the batch this thread fetches and parks; also the cluster it owns
      const uint8_t *ig = p.idx + (long long)g * p.N;
      unsigned int pre[kFitRedWarps + 1];   // prefix sums of the list lengths
      pre[0] = 0;
#pragma unroll
      for (int q = 0; q < kFitRedWarps; ++q) pre[q + 1] = pre[q] + (first ? 0u : lcnt[q]);
      const long long n_tot = first ? (r1 - r0) : (long long)pre[kFitRedWarps];
      const int nbat = (int)((n_tot + 255) / 256);
      if (p.clk && tid == 64) { p.clk[((long long)g * nx + bx) * 16 + 6] += n_tot; p.clk[((long long)g * nx + bx) * 16 + 7] += nbat; }
      auto buf_xd = [&](int b) { return reinterpret_cast<double2 *>(sgen + kFitSmemA + (b & 1) * kFitStageBytes); };              // [256][8] double2
      auto buf_cs = [&](int b) { return reinterpret_cast<double2 *>(sgen + kFitSmemA + (b & 1) * kFitStageBytes + 32768); };      // [256] {w, wn}
      auto buf_bm = [&](int b) { return reinterpret_cast<uint32_t *>(sgen + kFitSmemA + (b & 1) * kFitStageBytes + 36864); };     // [256][16]: 8 words "leaves", 8 words "joins"
      // entry: x = row - r0, y = k_old | k_new << 8 | pending << 17 (nothing here may consume the loaded value: it is still in flight)
      auto valid_entry = [&](int b) -> bool { return (long long)b * 256 + j < n_tot; };
      auto load_entry = [&](int b) -> uint2 {
        const long long f = (long long)b * 256 + j;
        if (f >= n_tot) return make_uint2(0u, 0u);
        if (first) return make_uint2((uint32_t)f, (1u << 17));
        int q = 0;
        unsigned int base = 0;
#pragma unroll
        for (int u = 1; u < kFitRedWarps; ++u)
          if (f >= (long long)pre[u]) { q = u; base = pre[u]; }
        return __ldcg(chg_cta + (long long)q * cap_w + (f - (long long)base));
      };
      uint4 xr[4];
      float wv = 0.f;
      double wnv = 0.0;
      int knv = 0;
      auto load_data = [&](const uint2 e, bool valid) {
        if (!valid) return;
        const long long rr = r0 + e.x, gr_ = (long long)g * p.N + rr;
        if (rows_bf16) {
          xr[0] = __ldg(reinterpret_cast<const uint4 *>(p.ahi + gr_ * kD));
          xr[1] = __ldg(reinterpret_cast<const uint4 *>(p.ahi + gr_ * kD) + 1);
        } else {
#pragma unroll
          for (int q4 = 0; q4 < 4; ++q4) xr[q4] = __ldg(reinterpret_cast<const uint4 *>(p.rows + gr_ * kD) + q4);
        }
        const long long tk_ = (msh >= 0) ? (rr >> msh) : (rr / p.M);
        wv = __ldg(p.wt + (long long)g * p.nf_tok + tk_);
        wnv = __ldg(p.wn + gr_);
        knv = (e.y & (1u << 17)) ? (int)__ldcg(ig + rr) : (int)((e.y >> 8) & 255u);
      };
      auto park = [&](int b, const uint2 e, bool valid) {
        if (!valid) return;
        const uint32_t ko = e.y & 255u;
        if (!first && (uint32_t)knv == ko) return;   // a queued row that stayed where it was
        float x[kD];
        if (rows_bf16) {
          const uint32_t u[8] = {xr[0].x, xr[0].y, xr[0].z, xr[0].w, xr[1].x, xr[1].y, xr[1].z, xr[1].w};
#pragma unroll
          for (int q8 = 0; q8 < 8; ++q8) { x[2 * q8] = __uint_as_float(u[q8] << 16); x[2 * q8 + 1] = __uint_as_float(u[q8] & 0xFFFF0000u); }
        } else {
#pragma unroll
          for (int q4 = 0; q4 < 4; ++q4) { x[4 * q4] = __uint_as_float(xr[q4].x); x[4 * q4 + 1] = __uint_as_float(xr[q4].y); x[4 * q4 + 2] = __uint_as_float(xr[q4].z); x[4 * q4 + 3] = __uint_as_float(xr[q4].w); }
        }
        double2 *xd = buf_xd(b) + j * 8;
#pragma unroll
        for (int q8 = 0; q8 < 8; ++q8) xd[q8] = make_double2((double)x[2 * q8], (double)x[2 * q8 + 1]);
        buf_cs(b)[j] = make_double2((double)wv, wnv);
        uint32_t *bm = buf_bm(b);
        if (!first) atomicOr(bm + ko * 16 + (j >> 5), 1u << (j & 31));
        atomicOr(bm + (uint32_t)knv * 16 + 8 + (j >> 5), 1u << (j & 31));
      };
      // this thread's cluster: sums in registers, in 16-byte chunks ROTATED by the lane (slot q holds chunk (q + lane) & 7) so that
      // the row reads of a warp (every lane another row, all lanes the same slot) fall into 8 different bank groups
      double2 aA[8], aB[8];
      double aW, aC;
      {
        const double2 *src = reinterpret_cast<const double2 *>(acc_s + j * kFitP);
#pragma unroll
        for (int q = 0; q < 8; ++q) { const int c = (q + lane) & 7; aA[q] = src[c]; aB[q] = src[8 + c]; }
        aW = acc_s[j * kFitP + 2 * kD]; aC = acc_s[j * kFitP + 2 * kD + 1];
      }
      for (int e = j; e < 2 * 256 * 16; e += 256) reinterpret_cast<uint32_t *>(sgen + kFitSmemA + (e >> 12) * kFitStageBytes + 36864)[e & 4095] = 0u;
      asm volatile("bar.sync 1, 256;" ::: "memory");
      uint2 e_cur = load_entry(0), e_nxt = load_entry(1);
      load_data(e_cur, valid_entry(0));
      park(0, e_cur, valid_entry(0));
      asm volatile("bar.sync 1, 256;" ::: "memory");
      for (int b = 0; b < nbat; ++b) {
        if (b + 1 < nbat) load_data(e_nxt, valid_entry(b + 1));   // batch b + 1: rows and weights in flight
        const uint2 e_nn = (b + 2 < nbat) ? load_entry(b + 2) : make_uint2(0u, 0u);   // batch b + 2: its list entries
        {
          const double2 *xd = buf_xd(b);
          const double2 *cs = buf_cs(b);
          uint32_t *bm = buf_bm(b) + j * 16;
          uint32_t nz = 0;   // non-empty words of my bitmap row: bits 0-7 "leaves", 8-15 "joins"
          {
            const uint4 w0 = reinterpret_cast<const uint4 *>(bm)[0], w1 = reinterpret_cast<const uint4 *>(bm)[1];
            const uint4 w2 = reinterpret_cast<const uint4 *>(bm)[2], w3 = reinterpret_cast<const uint4 *>(bm)[3];
            const uint32_t ww[16] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w, w2.x, w2.y, w2.z, w2.w, w3.x, w3.y, w3.z, w3.w};
#pragma unroll
            for (int q = 0; q < 16; ++q) nz |= (ww[q] != 0u) ? (1u << q) : 0u;
          }
          uint32_t word = 0;
          int wi = 0;
          for (;;) {
            if (word == 0u) {
              if (nz == 0u) break;
              wi = __ffs(nz) - 1;
              nz &= nz - 1;
              word = bm[wi];
              bm[wi] = 0u;   // the bitmap is clean again for the batch after next
            }
            const int e = (wi & 7) * 32 + (__ffs(word) - 1);
            word &= word - 1;
            double2 c2 = cs[e];
            if (wi < 8) { c2.x = -c2.x; c2.y = -c2.y; }
            const double2 *xe = xd + e * 8;
            double2 xv[8];   // all eight loads in flight before the first use (the compiler would otherwise chain them through one register quad)
#pragma unroll
            for (int q = 0; q < 8; ++q) xv[q] = xe[(q + lane) & 7];
            asm volatile("" ::: "memory");
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              aA[q].x = fma(c2.x, xv[q].x, aA[q].x); aA[q].y = fma(c2.x, xv[q].y, aA[q].y);
              aB[q].x = fma(c2.y, xv[q].x, aB[q].x); aB[q].y = fma(c2.y, xv[q].y, aB[q].y);
            }
            aW += c2.x;
            aC += (wi < 8) ? -1.0 : 1.0;
          }
        }
        if (b + 1 < nbat) park(b + 1, e_nxt, valid_entry(b + 1));
        e_nxt = e_nn;
        asm volatile("bar.sync 1, 256;" ::: "memory");
      }
      {
        double2 *dst = reinterpret_cast<double2 *>(acc_s + j * kFitP);
#pragma unroll
        for (int q = 0; q < 8; ++q) { const int c = (q + lane) & 7; dst[c] = aA[q]; dst[8 + c] = aB[q]; }
        acc_s[j * kFitP + 2 * kD] = aW; acc_s[j * kFitP + 2 * kD + 1] = aC;
      }
      fence_proxy_async();   // generic-proxy use of the scoring buffers ends here; the next pass's TMA / tensor core use them again
    }
    __syncthreads();
    if (p.clk && tid == 0 && first) p.clk[((long long)g * nx + bx) * 16 + 8] += clock64() - clk_last;
    // publish this CTA's sums: record k = A[16] | B[16] | W | cnt
    {
      double2 *dst = reinterpret_cast<double2 *>(p.part + ((long long)g * nx + bx) * kN * kFitP);
      const double2 *src = reinterpret_cast<const double2 *>(acc_s);
      for (int e = tid; e < kN * kFitP / 2; e += kThreads) dst[e] = src[e];
    }
    clk_mark(2);

    // ---------------- (d) every CTA of the group has published its partials ----------------
    ++epoch;
    group_barrier(p.bar + g, epoch * (unsigned int)nx, stg);
    if (tid == 0) {
      misc[0] = (stg && !p.skip_scoring) ? __ldcg(&stg->changed[t]) : 1;
      misc[1] = fit_lost(stg) ? 1 : 0;
    }
    __syncthreads();
    if (misc[1]) break;   // a CTA of the group was lost: the partials are incomplete, leave the codebook as it is
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
    if (tid == 0) misc[1] = fit_lost(stg) ? 1 : 0;
    __syncthreads();
    if (misc[1]) break;
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
