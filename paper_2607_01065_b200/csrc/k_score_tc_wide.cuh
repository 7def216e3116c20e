// k_score_tc_wide.cuh -- tcgen05 scoring + fused arg-max for wide sub-vectors, d = 64 KB (KB = 1, 2: d = 64, 128), K <= 256:
// the paper's own operating point D = 128, where one score costs 256 tensor flops and the tensor pipe,
// not the arg-max epilogue, is the limiter.
//
// Same numerics as k_score_tc.cuh: per 128-row tile and 16-column K step
//     D += A_hi . B_hi^T + A_hi . B_lo^T (+ A_lo . B_hi^T when the rows are not bf16-exact),   then   D += 1 . B_bias^T,
// fp32 accumulation in TMEM, so D[i][k] ~= 2 g_k r_i.s_k - g_k^2 (Eq. 5) within a bound E_i; the epilogue is the
// same max / arg-max (tile_argmax); a row whose top-2 gap is within the bound goes to a list and is decided by the exact
// fp64 kernel (k_wide_assign, list mode).  The N x K score matrix never leaves the SM.
//
// Operands are K-major SWIZZLE_128B tiles: a shared-memory row holds 64 bf16 (one "K block"), d = 128 is two K blocks.
// Shared memory: B_hi and B_lo of the whole codebook (KB x 32 KB each, loaded once per CTA), the bias image and the
// constant tile (SWIZZLE_32B, K = 16), and a ring of 2 slots of ONE K block of A (hi and lo plane, 16 KB each): the TMA
// refills a slot for the next tile while the MMAs of the other K block run.  2 x 256 TMEM columns: tile i's epilogue
// overlaps tile i+1's MMAs.  Warp roles as in k_score_tc: warp 0 TMA, warp 1 MMA issue, warps 2-9 epilogue.
#pragma once
#include "k_score_tc.cuh"

namespace gsrq {
namespace tc {

constexpr uint32_t kWKbBytesA = kTileM * 128;   // one K block of one A plane: 128 rows x 128 B
constexpr uint32_t kWKbBytesB = kN * 128;       // one K block of one B plane: 256 rows x 128 B
constexpr int kWSlots = 2;

template <int KB> struct WideSmem {
  static constexpr uint32_t kB = 0;                                   // [hi | lo][KB] K blocks of B
  static constexpr uint32_t kBias = 2 * KB * kWKbBytesB;               // bias image (SWIZZLE_32B)
  static constexpr uint32_t kOnes = kBias + kBImgBytes;                // constant A_1 tile (SWIZZLE_32B)
  static constexpr uint32_t kA = kOnes + kPlaneBytes;                  // ring: kWSlots x {hi, lo} K blocks of A
  static constexpr uint32_t kBar = kA + kWSlots * 2 * kWKbBytesA;
  static constexpr uint32_t kTotal = kBar + 256 + 1024;
};
static_assert(WideSmem<2>::kA % 1024 == 0 && WideSmem<2>::kTotal <= 227 * 1024, "shared-memory budget / SWIZZLE_128B alignment");

struct ScoreWideParams {
  const uint8_t *bimg;    // [G]{B_hi[KB][32 KB], B_lo[KB][32 KB], bias[8 KB]} operand images
  const int *gmax;        // [G] bit pattern of max_k g_k (mode 0)
  const float *rnorm;     // [G][N]
  const float *gains;     // stage slice
  long long cb_stride_g;
  uint8_t *idx;           // [G][N]
  long long N;
  int n_tiles, n_planes, K, mode;
  DevStats *st;
  int slot;
  uint2 *list;            // undecided rows {g*N + i, mask of the candidate 16-codeword groups} for the exact kernel
  unsigned int *list_cnt;
  float *dbg;             // optional [G][N][256] raw scores (tests)
};

// K-major SWIZZLE_128B descriptor: rows of 128 B, 8-row groups 1024 B apart; layout code 2.
__device__ __forceinline__ uint64_t make_desc_sw128(uint32_t saddr) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// byte offset of element (row, col) of one K block ([rows][64] bf16) in the SWIZZLE_128B layout
__host__ __device__ __forceinline__ uint32_t sw128_off(int row, int col) {
  return (uint32_t)row * 128u + (((((uint32_t)col >> 3) ^ ((uint32_t)row & 7u)) & 7u) << 4) + ((uint32_t)col & 7u) * 2u;
}

template <int KB> __host__ __device__ constexpr uint32_t wide_bimg_bytes() { return 2 * KB * kWKbBytesB + kBImgBytes; }

// Operand images of one (group, stage slice): c' = fl32(2 fl32(g_k s_kj)) split hi / lo, bias b = fl32(g_k^2) split in three
// (mode 1, projection: c' = 2 s_kj, b = 0); rows k >= K can never win.  grid = (G, 8): 32 codewords per CTA, block = 256;
// gmax[g] (zeroed by the caller) receives the bit pattern of max_k g_k.
template <int KB>
__global__ void __launch_bounds__(256) k_bimg_wide(const float *__restrict__ shapes, const float *__restrict__ gains, long long cb_stride_g,
                                                   int K, int mode, uint8_t *__restrict__ bimg, int *__restrict__ gmax) {
  const int g = blockIdx.x, k0 = blockIdx.y * 32;
  constexpr int d = 64 * KB;
  uint8_t *img = bimg + (size_t)g * wide_bimg_bytes<KB>();
  for (int e = threadIdx.x; e < 32 * d; e += 256) {   // coalesced over the codeword rows
    const int k = k0 + e / d, j = e % d;
    const bool dead = k >= K;
    float c = 0.f;
    if (!dead) {
      const float sj = shapes[((long long)g * cb_stride_g + k) * d + j];
      c = (mode == 0) ? 2.0f * __fmul_rn(gains[(long long)g * cb_stride_g + k], sj) : 2.0f * sj;
    }
    const __nv_bfloat16 hi = __float2bfloat16_rn(c);
    const __nv_bfloat16 lo = __float2bfloat16_rn(__fsub_rn(c, __bfloat162float(hi)));
    const uint32_t off = (uint32_t)(j >> 6) * kWKbBytesB + sw128_off(k, j & 63);
    *reinterpret_cast<__nv_bfloat16 *>(img + off) = hi;
    *reinterpret_cast<__nv_bfloat16 *>(img + KB * kWKbBytesB + off) = lo;
  }
  if (threadIdx.x < 32) {
    const int k = k0 + threadIdx.x;
    const bool dead = k >= K;
    const float gk = (!dead && mode == 0) ? gains[(long long)g * cb_stride_g + k] : 1.0f;
    const float b = dead ? 3.0e38f : ((mode == 0) ? __fmul_rn(gk, gk) : 0.0f);
    const __nv_bfloat16 b1 = __float2bfloat16_rn(b);
    const float r1 = __fsub_rn(b, __bfloat162float(b1));
    const __nv_bfloat16 b2 = __float2bfloat16_rn(r1);
    const __nv_bfloat16 b3 = __float2bfloat16_rn(__fsub_rn(r1, __bfloat162float(b2)));
    uint8_t *bias = img + 2 * KB * kWKbBytesB;
    for (int j = 0; j < kD; ++j) {
      __nv_bfloat16 v = __float2bfloat16_rn(0.f);
      if (j == 0) v = __hneg(b1);
      if (j == 1) v = __hneg(b2);
      if (j == 2) v = __hneg(b3);
      *reinterpret_cast<__nv_bfloat16 *>(bias + sw32_off(k, j)) = v;
    }
    if (!dead && mode == 0 && gmax) atomicMax(gmax + g, __float_as_int(fmaxf(gk, 0.f)));
  }
}

template <int KB, bool DBG>
__global__ void __launch_bounds__(kThreads, 1)
k_score_tc_wide(const __grid_constant__ CUtensorMap tm_hi, const __grid_constant__ CUtensorMap tm_lo, ScoreWideParams p) {
  using L = WideSmem<KB>;
  extern __shared__ uint8_t smem_raw[];
  const int g = blockIdx.y;
  if (group_done(p.st, g, p.slot)) return;
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *sgen = smem_raw + (sbase - smem_u32(smem_raw));
  const uint32_t bar0 = sbase + L::kBar;
  auto full_a = [&](int s) { return bar0 + 8u * s; };
  auto empty_a = [&](int s) { return bar0 + 8u * (kWSlots + s); };
  auto tmem_full = [&](int b) { return bar0 + 8u * (2 * kWSlots + b); };
  auto tmem_empty = [&](int b) { return bar0 + 8u * (2 * kWSlots + 2 + b); };
  const uint32_t b_full = bar0 + 8u * (2 * kWSlots + 4);
  volatile uint32_t *tmem_slot = reinterpret_cast<volatile uint32_t *>(sgen + L::kBar + 8 * (2 * kWSlots + 5));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kWSlots; ++s) { mbar_init(full_a(s), 1); mbar_init(empty_a(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tmem_full(b), 1); mbar_init(tmem_empty(b), 4); }
    mbar_init(b_full, 1);
    fence_barrier_init();
  }
  for (int e = threadIdx.x; e < kTileM * kD; e += kThreads) {   // constant A_1 tile: columns 0,1,2 = 1.0
    const int row = e >> 4, col = e & 15;
    *reinterpret_cast<uint16_t *>(sgen + L::kOnes + sw32_off(row, col)) = (col < 3) ? 0x3F80 : 0;
  }
  fence_proxy_async();
  if (warp == 1) tmem_alloc(smem_u32((const void *)tmem_slot), 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const int n_my = (p.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;

  if (warp == 0) {
    if (lane == 0) {
      mbar_expect_tx(b_full, wide_bimg_bytes<KB>());
      const uint8_t *src = p.bimg + (size_t)g * wide_bimg_bytes<KB>();
      // one bulk copy per 32 KB K block (and the bias image)
      for (int c = 0; c < 2 * KB; ++c) bulk_g2s(sbase + L::kB + c * kWKbBytesB, src + (size_t)c * kWKbBytesB, kWKbBytesB, b_full);
      bulk_g2s(sbase + L::kBias, src + (size_t)2 * KB * kWKbBytesB, kBImgBytes, b_full);
      for (int it = 0; it < n_my; ++it) {
        const int tile = blockIdx.x + it * gridDim.x;
        for (int kb = 0; kb < KB; ++kb) {
          const int u = it * KB + kb, sl = u % kWSlots, ph = (u / kWSlots) & 1;
          mbar_wait(empty_a(sl), ph ^ 1);
          mbar_expect_tx(full_a(sl), p.n_planes * kWKbBytesA);
          tma_load_3d(sbase + L::kA + sl * 2 * kWKbBytesA, &tm_hi, kb * 64, tile * kTileM, g, full_a(sl));
          if (p.n_planes == 2) tma_load_3d(sbase + L::kA + sl * 2 * kWKbBytesA + kWKbBytesA, &tm_lo, kb * 64, tile * kTileM, g, full_a(sl));
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      const uint64_t d_bias = make_desc_sw32(sbase + L::kBias), d_ones = make_desc_sw32(sbase + L::kOnes);
      mbar_wait(b_full, 0);
      for (int it = 0; it < n_my; ++it) {
        const int buf = it & 1, bph = (it >> 1) & 1;
        mbar_wait(tmem_empty(buf), bph ^ 1);
        const uint32_t dacc = tmem_base + buf * kN;
        for (int kb = 0; kb < KB; ++kb) {
          const int u = it * KB + kb, sl = u % kWSlots, ph = (u / kWSlots) & 1;
          mbar_wait(full_a(sl), ph);
          tc_fence_after();
          const uint32_t a_hi = sbase + L::kA + sl * 2 * kWKbBytesA, a_lo = a_hi + kWKbBytesA;
          const uint32_t b_hi = sbase + L::kB + kb * kWKbBytesB, b_lo = b_hi + KB * kWKbBytesB;
#pragma unroll
          for (int ks = 0; ks < 4; ++ks) {   // 16 bf16 = 32 bytes per K step inside the 128-byte swizzled row
            const uint64_t dah = make_desc_sw128(a_hi + ks * 32), dbh = make_desc_sw128(b_hi + ks * 32), dbl = make_desc_sw128(b_lo + ks * 32);
            mma_f16(dacc, dah, dbh, kIdesc, (kb | ks) ? 1u : 0u);
            mma_f16(dacc, dah, dbl, kIdesc, 1);
            if (p.n_planes == 2) mma_f16(dacc, make_desc_sw128(a_lo + ks * 32), dbh, kIdesc, 1);
          }
          mma_commit(empty_a(sl));
        }
        mma_f16(dacc, d_ones, d_bias, kIdesc, 1);
        mma_commit(tmem_full(buf));
      }
    }
  } else {
    const int q = warp & 3;        // TMEM lane quarter this warp may access
    const int wg = (warp - 2) >> 2;
    const float gm = (p.mode == 0) ? __int_as_float(p.gmax[g]) : 1.0f;
    // error bound of a score with gain g:  E(g) = rho 2^-17 (2 g ||r||) + 2^-18 g^2.  In units of
    // 2^-17 (2 g ||r||): operand splits 0.5 each, dropped lo.lo 0.5, 4-bit index packing 0.25, fp32 accumulation of 3 d + 3 products.
    // The tensor core's accumulation is not specified as round-to-nearest: each step is budgeted at 2^-23 (truncation / alignment
    // loss), i.e. 6.0 units at d = 128 and 3.0 at d = 64.
    // rho = 8 / 9 (d = 128, one / two operand planes), 5.5 / 6.5 (d = 64); measured worst error: 1.3 / 1.7 units (tests/test_gpu_wide.py)
    const float rho17 = (KB == 2 ? (p.n_planes == 1 ? 8.0f : 9.0f) : (p.n_planes == 1 ? 5.5f : 6.5f)) * 7.62939453125e-6f;
    unsigned int n_changed = 0;
    for (int it = wg; it < n_my; it += 2) {
      const int buf = wg, bph = (it >> 1) & 1;
      const int tile = blockIdx.x + it * gridDim.x;
      const long long row = (long long)tile * kTileM + q * 32 + lane;
      const long long gr = (long long)g * p.N + row;
      float rn = 0.f;
      uint8_t k_old = 0;
      if (row < p.N) { rn = p.rnorm[gr]; k_old = p.idx[gr]; }
      mbar_wait(tmem_full(buf), bph);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + buf * kN;
      float gmA[16], best, second;
      int gi, ji;
      tile_argmax<DBG>(taddr, gmA, best, second, gi, ji, (DBG && row < p.N) ? p.dbg + gr * kN : nullptr, [&]() {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tmem_empty(buf));
      });
      const int k_new = gi * 16 + ji;
      const float gk = __ldg(p.gains + (long long)g * p.cb_stride_g + min(k_new, p.K - 1));
      const float E2 = decision_margin(best, rn, gk, gm, rho17, p.mode);
      if (row < p.N) {
        if (best - second <= E2) {
          p.list[atomicAdd(p.list_cnt, 1u)] = make_uint2((uint32_t)gr, candidate_groups(gmA, best, E2));   // the exact kernel decides (and counts the change)
        } else {
          n_changed += (k_old != (uint8_t)k_new);
          p.idx[gr] = (uint8_t)k_new;
        }
      }
    }
    if (p.st) {
      for (int off = 16; off; off >>= 1) n_changed += __shfl_xor_sync(0xffffffffu, n_changed, off);
      if (lane == 0 && n_changed) atomicAdd(reinterpret_cast<unsigned long long *>(&p.st[g].changed[p.slot]), (unsigned long long)n_changed);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, 512);
}

}  // namespace tc
}  // namespace gsrq
