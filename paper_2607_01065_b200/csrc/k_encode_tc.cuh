// k_encode_tc.cuh -- fused multi-stage residual-quantization encode on the tcgen05 tensor cores
// (RQ; assignment Eq. 5).  d = 16, K <= 256, stages [0, n_stages),
// n_stages <= kEncMaxS, bf16 input read straight from the KV tensor by TMA.
//
// A 128-row tile goes through all stages without leaving the SM:
//   stage 0:  D = X.B_hi^T + X.B_lo^T + 1.B_bias^T          X = the bf16 rows themselves (exact operand)
//   epilogue: k = arg-max (tile_argmax), code byte out, r <- fl32(r - fl32(g_k s_k)) in registers
//             (fp32, element-wise, no FMA contraction: DESIGN.md reading c-P), then the operand planes
//             of the residual, R_hi = bf16(r), R_lo = bf16(r - R_hi), go back to shared memory
//   stage s:  D = R_hi.B_hi^T + R_hi.B_lo^T + R_lo.B_hi^T + 1.B_bias^T   against stage s's images
// The N x K score matrix and the residual between stages are never written to HBM; optionally the
// final fp32 residual is.  A row whose top-2 gap is within the filter's error bound at any stage is
// handed, with its candidate codeword groups, to the exact CUDA-core path (k_encode_exact), which takes
// the row over from that stage.
//
// Warp roles (320 threads, one CTA per SM, persistent over tiles of one group): warp 0 TMA producer,
// warp 1 tcgen05.mma issue, warps 2-5 / 6-9 two epilogue warpgroups, each owning one 256-column
// TMEM accumulator and every other tile of the CTA, so that one tile's epilogue overlaps the
// other's MMAs.
#pragma once
#include "k_score_tc.cuh"

namespace gsrq {
namespace tc {

constexpr int kEncMaxS = 4;     // stages per fused pass (shared-memory budget: 24 KB of images per stage)
constexpr int kEncStages = 4;   // TMA ring depth for the stage-0 tiles
constexpr uint32_t kEncSmemOnes = kEncMaxS * 3 * kBImgBytes;                 // 98304
constexpr uint32_t kEncSmemA = kEncSmemOnes + kPlaneBytes;                   // ring of kEncStages tiles
constexpr uint32_t kEncSmemP = kEncSmemA + kEncStages * kPlaneBytes;         // residual planes [2 buffers][hi, lo]
constexpr uint32_t kEncSmemBar = kEncSmemP + 4 * kPlaneBytes;
constexpr uint32_t kEncSmemCb = kEncSmemBar + 256;                           // fp32 codebook of the pass's stages: [stage]{shapes [256][16], gains [256]}
constexpr uint32_t kEncCbStage = kN * kD * 4 + kN * 4;
constexpr uint32_t kEncSmemTotal = kEncSmemCb + kEncMaxS * kEncCbStage + 1024;   // + alignment slack
static_assert(kEncSmemTotal <= 227 * 1024, "shared-memory budget");

struct EncTcParams {
  const uint8_t *bimg;     // [G][n_stages][3][8192] operand images (mode 0)
  const int *gmax;         // [G][n_stages] bit pattern of max_k g_k
  const float *shapes;     // [G][S][K][16]
  const float *gains;      // [G][S][K]
  int S, K, n_stages;      // cb->S, K, stages of this pass
  int s0;                  // first stage of this pass (absolute index into the codebook / code planes)
  const float *res_in;     // FROM_ROWS: [G][N][16] fp32 rows the pass starts from (may alias res_out)
  uint8_t *codes;          // plane s, group g, row i at codes[s*code_stride_s + g*N + i]; nullptr: no codes wanted
  long long code_stride_s;
  float *res_out;          // [G][N][16] or nullptr
  long long N;             // rows per group
  int n_tiles;
  uint2 *list;             // rows for the exact path: {g*N + i, candidate-group mask | stage << 16}
  unsigned int *list_cnt;
};

__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, int c2, int c3, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(dst),
      "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}

// tm_kv: 4-D map over the KV tensor {16 (contiguous), M, T, G} ({16, M, G, T} when head_inner), box {16, M, 128 / M, 1}, SWIZZLE_32B:
// one box is the 128 consecutive rows (t, m) of a tile, laid out as the K-major A operand.
// FROM_ROWS = false: stage s0 = 0 reads the bf16 rows of the KV tensor through tm_kv (exact single-plane operand).
// FROM_ROWS = true : the pass starts from fp32 rows (a residual, or an fp32 tensor): the epilogue loads them, builds the
//                    two operand planes itself and every stage runs the two-plane MMAs; tm_kv is unused.
template <bool FROM_ROWS>
__global__ void __launch_bounds__(kThreads, 1) k_encode_tc(const __grid_constant__ CUtensorMap tm_kv, EncTcParams p, int tok_per_tile,
                                                                  int head_inner) {
  extern __shared__ uint8_t smem_raw[];
  const int g = blockIdx.y;
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *sgen = smem_raw + (sbase - smem_u32(smem_raw));
  const uint32_t bar0 = sbase + kEncSmemBar;
  auto full_a = [&](int s) { return bar0 + 8u * s; };
  auto empty_a = [&](int s) { return bar0 + 8u * (kEncStages + s); };
  auto tmem_full = [&](int b) { return bar0 + 8u * (2 * kEncStages + b); };
  auto tmem_empty = [&](int b) { return bar0 + 8u * (2 * kEncStages + 2 + b); };
  auto planes_ready = [&](int b) { return bar0 + 8u * (2 * kEncStages + 4 + b); };
  const uint32_t b_full = bar0 + 8u * (2 * kEncStages + 6);
  volatile uint32_t *tmem_slot = reinterpret_cast<volatile uint32_t *>(sgen + kEncSmemBar + 8 * (2 * kEncStages + 7));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int S = p.n_stages;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kEncStages; ++s) { mbar_init(full_a(s), 1); mbar_init(empty_a(s), 4); }
    for (int b = 0; b < 2; ++b) { mbar_init(tmem_full(b), 1); mbar_init(tmem_empty(b), 4); mbar_init(planes_ready(b), 4); }
    mbar_init(b_full, 1);
    fence_barrier_init();
  }
  // constant A_1 tile: columns 0,1,2 = 1.0 (bf16 0x3F80), rest 0
  for (int e = threadIdx.x; e < kTileM * kD; e += kThreads) {
    const int row = e >> 4, col = e & 15;
    *reinterpret_cast<uint16_t *>(sgen + kEncSmemOnes + sw32_off(row, col)) = (col < 3) ? 0x3F80 : 0;
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
      mbar_expect_tx(b_full, (uint32_t)S * 3 * kBImgBytes);
      bulk_g2s(sbase, p.bimg + (size_t)g * S * 3 * kBImgBytes, (uint32_t)S * 3 * kBImgBytes, b_full);
      for (int it = 0; it < (FROM_ROWS ? 0 : n_my); ++it) {
        const int st = it % kEncStages, ph = (it / kEncStages) & 1;
        const int tile = blockIdx.x + it * gridDim.x;
        mbar_wait(empty_a(st), ph ^ 1);
        mbar_expect_tx(full_a(st), kPlaneBytes);
        const int tok0 = tile * tok_per_tile;
        tma_load_4d(sbase + kEncSmemA + st * kPlaneBytes, &tm_kv, 0, 0, head_inner ? g : tok0, head_inner ? tok0 : g, full_a(st));
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      const uint64_t d_ones = make_desc_sw32(sbase + kEncSmemOnes);
      mbar_wait(b_full, 0);
      // static schedule: tiles in pairs (one per accumulator / epilogue warpgroup), stage by stage
      for (int pr = 0; 2 * pr < n_my; ++pr) {
        for (int s = 0; s < S; ++s) {
          const uint64_t d_bhi = make_desc_sw32(sbase + (uint32_t)s * 3 * kBImgBytes);
          const uint64_t d_blo = make_desc_sw32(sbase + (uint32_t)s * 3 * kBImgBytes + kBImgBytes);
          const uint64_t d_bias = make_desc_sw32(sbase + (uint32_t)s * 3 * kBImgBytes + 2 * kBImgBytes);
          for (int b = 0; b < 2; ++b) {
            const int it = 2 * pr + b;
            if (it >= n_my) continue;
            const uint32_t d = tmem_base + b * kN;
            if (s == 0 && !FROM_ROWS) {
              const int st = it % kEncStages, ph = (it / kEncStages) & 1;
              mbar_wait(tmem_empty(b), (pr & 1) ^ 1);
              mbar_wait(full_a(st), ph);
              tc_fence_after();
              const uint64_t d_a = make_desc_sw32(sbase + kEncSmemA + st * kPlaneBytes);
              mma_f16(d, d_a, d_bhi, kIdesc, 0);
              mma_f16(d, d_a, d_blo, kIdesc, 1);
            } else {
              if (FROM_ROWS && s == 0) mbar_wait(tmem_empty(b), (pr & 1) ^ 1);
              mbar_wait(planes_ready(b), FROM_ROWS ? (uint32_t)((pr * S + s) & 1) : (uint32_t)((pr * (S - 1) + (s - 1)) & 1));
              tc_fence_after();
              const uint64_t d_hi = make_desc_sw32(sbase + kEncSmemP + (2 * b) * kPlaneBytes);
              const uint64_t d_lo = make_desc_sw32(sbase + kEncSmemP + (2 * b + 1) * kPlaneBytes);
              mma_f16(d, d_hi, d_bhi, kIdesc, 0);
              mma_f16(d, d_hi, d_blo, kIdesc, 1);
              mma_f16(d, d_lo, d_bhi, kIdesc, 1);
            }
            mma_f16(d, d_ones, d_bias, kIdesc, 1);
            mma_commit(tmem_full(b));
          }
        }
      }
    }
  } else {
    // Epilogue: warpgroup wg owns accumulator wg and the CTA's tiles it = wg, wg + 2, ...; thread = row.
    const int q = warp & 3;  // TMEM lane quarter this warp may access
    const int wg = (warp - 2) >> 2;
    const int r_in_tile = q * 32 + lane;
    uint8_t *planes = sgen + kEncSmemP + (2 * wg) * kPlaneBytes;
    const uint32_t sw = ((uint32_t)(r_in_tile >> 2) & 1u) << 4;  // SWIZZLE_32B: the two 16-byte chunks of a row swap
    // the fp32 codebook of the pass's stages -> shared memory: the gain (decision margin) and the codeword (subtraction) of a row's
    // winner sit on the critical path between a tile's stages, and a global load there costs ten times a shared-memory one
    {
      const int et = threadIdx.x - 64;  // 0..255
      for (int s = 0; s < S; ++s) {
        float *cbs = reinterpret_cast<float *>(sgen + kEncSmemCb + s * kEncCbStage);
        const long long c0 = ((long long)g * p.S + p.s0 + s) * p.K;
        const float4 *src = reinterpret_cast<const float4 *>(p.shapes + c0 * kD);
        for (int e = et; e < p.K * (kD / 4); e += 256) reinterpret_cast<float4 *>(cbs)[e] = __ldg(src + e);
        if (et < p.K) cbs[kN * kD + et] = __ldg(p.gains + c0 + et);
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");
    }
    for (int it = wg; it < n_my; it += 2) {
      const int pr = it >> 1;
      const int st = it % kEncStages, ph = (it / kEncStages) & 1;
      const int tile = blockIdx.x + it * gridDim.x;
      const long long row = (long long)tile * kTileM + r_in_tile;
      const long long gr = (long long)g * p.N + row;
      bool alive = row < p.N;
      float r[kD];
      auto publish_planes = [&]() {  // operand planes of r for the next MMAs: R_hi = bf16(r), R_lo = bf16(r - R_hi)
        uint32_t h[8], l[8];
#pragma unroll
        for (int j = 0; j < kD; j += 2) {  // one packed conversion per pair; the high half is re-read by masking
          const __nv_bfloat162 hp = __floats2bfloat162_rn(r[j], r[j + 1]);
          h[j / 2] = *reinterpret_cast<const uint32_t *>(&hp);
          const float d0 = __fsub_rn(r[j], __uint_as_float(h[j / 2] << 16));
          const float d1 = __fsub_rn(r[j + 1], __uint_as_float(h[j / 2] & 0xFFFF0000u));
          const __nv_bfloat162 lp = __floats2bfloat162_rn(d0, d1);
          l[j / 2] = *reinterpret_cast<const uint32_t *>(&lp);
        }
        uint8_t *ph_ = planes + r_in_tile * 32, *pl_ = planes + kPlaneBytes + r_in_tile * 32;
        *reinterpret_cast<uint4 *>(ph_ + (0u ^ sw)) = make_uint4(h[0], h[1], h[2], h[3]);
        *reinterpret_cast<uint4 *>(ph_ + (16u ^ sw)) = make_uint4(h[4], h[5], h[6], h[7]);
        *reinterpret_cast<uint4 *>(pl_ + (0u ^ sw)) = make_uint4(l[0], l[1], l[2], l[3]);
        *reinterpret_cast<uint4 *>(pl_ + (16u ^ sw)) = make_uint4(l[4], l[5], l[6], l[7]);
        fence_proxy_async();   // generic-proxy writes -> visible to the tensor core's async proxy
        tc_fence_before();     // this stage's tcgen05.ld is complete before the next MMAs overwrite the accumulator
        __syncwarp();
        if (lane == 0) mbar_arrive(planes_ready(wg));
      };
      for (int s = 0; s < S; ++s) {
        if (s == 0 && FROM_ROWS) {  // the pass starts from fp32 rows
          if (row < p.N) load_row_f32<kD>(p.res_in, gr, r);
          else {
#pragma unroll
            for (int j = 0; j < kD; ++j) r[j] = 0.0f;
          }
          publish_planes();
        } else if (s == 0) {  // the row itself, from the TMA-staged tile (exact bf16 -> fp32)
          mbar_wait(full_a(st), ph);
          const uint8_t *ar = sgen + kEncSmemA + st * kPlaneBytes + r_in_tile * 32;
          const uint4 c0 = *reinterpret_cast<const uint4 *>(ar + (0u ^ sw));
          const uint4 c1 = *reinterpret_cast<const uint4 *>(ar + (16u ^ sw));
          const uint32_t u[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            r[2 * e] = __uint_as_float(u[e] << 16);
            r[2 * e + 1] = __uint_as_float(u[e] & 0xFFFF0000u);
          }
        }
        float n2 = 0.0f;
#pragma unroll
        for (int j = 0; j < kD; ++j) n2 = fmaf(r[j], r[j], n2);
        const float rn = sqrtf(n2) * 1.00001f;  // upper bound of ||r||
        const float gm = __int_as_float(p.gmax[g * S + s]);
        const float rho17 = ((s == 0 && !FROM_ROWS) ? 2.0f : 4.5f) * 7.62939453125e-6f;  // rho 2^-17: one / two operand planes
        mbar_wait(tmem_full(wg), (uint32_t)((pr * S + s) & 1));
        tc_fence_after();
        if (s == 0 && !FROM_ROWS) {  // stage-0 MMAs are done with the tile and this warp has its rows: free the ring slot
          __syncwarp();
          if (lane == 0) mbar_arrive(empty_a(st));
        }
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + wg * kN;
        float gmA[16], best, second;
        int gi, ji;
        tile_argmax<false>(taddr, gmA, best, second, gi, ji, nullptr, [&]() {
          if (s == S - 1) {  // last stage of the tile: the accumulator is free for the next tile's stage 0
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tmem_empty(wg));
          }
        });
        const int k = gi * 16 + ji;
        const float *cbs = reinterpret_cast<const float *>(sgen + kEncSmemCb + s * kEncCbStage);
        const int kc = min(k, p.K - 1);
        const float gk = cbs[kN * kD + kc];
        const float E2 = decision_margin(best, rn, gk, gm, rho17, 0);
        if (alive && best - second <= E2) {  // ambiguous: the exact path takes the row over from this stage
          const uint32_t gmask = candidate_groups(gmA, best, E2);  // groups of 16 columns within the margin: the only candidates
          const unsigned int pos = atomicAdd(p.list_cnt, 1u);
          // without a code plane the decided stages of this pass cannot be replayed: the exact path restarts the pass
          p.list[pos] = p.codes ? make_uint2((uint32_t)gr, gmask | ((uint32_t)(p.s0 + s) << 16))
                                : make_uint2((uint32_t)gr, 0xFFFFu | ((uint32_t)p.s0 << 16));
          alive = false;
        }
        if (alive && p.codes) p.codes[(long long)(p.s0 + s) * p.code_stride_s + gr] = (uint8_t)k;
        // r <- fl32(r - fl32(g_k s_k)): the codeword comes from the fp32 codebook in shared memory
        const float4 *sp = reinterpret_cast<const float4 *>(cbs + kc * kD);
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const float4 sv = sp[v];
          r[4 * v] = __fsub_rn(r[4 * v], __fmul_rn(gk, sv.x));
          r[4 * v + 1] = __fsub_rn(r[4 * v + 1], __fmul_rn(gk, sv.y));
          r[4 * v + 2] = __fsub_rn(r[4 * v + 2], __fmul_rn(gk, sv.z));
          r[4 * v + 3] = __fsub_rn(r[4 * v + 3], __fmul_rn(gk, sv.w));
        }
        if (s + 1 < S) {  // operand planes of the residual for the next stage
          publish_planes();
        } else if (alive && p.res_out) {
          store_row_f32<kD>(p.res_out, gr, r);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, 512);
}

}  // namespace tc
}  // namespace gsrq
