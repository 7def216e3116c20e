// k_attn.cuh -- decode-attention straight from the GSRQ codes (PAPER.md:443 (ii): "on-the-fly bit-unpacking, dequantization,
// RoPE, and attention computation during decoding without materializing intermediate FP16 tensors"; the step is
// bound by memory traffic, and the codes are 16x smaller than the bf16 cache at 1 bit per element).
//
// For sequence b, KV head g and its n_rep = Hq / G query heads (grouped-query attention; LLaMA-3-8B: 32 / 8), over the
// sequence's tokens t:      out_h = sum_t softmax_t(scale q_h . k_t) vhat_t,
//     khat_t = sum_s cK^(s)[aK^(s)_t],  vhat_t = sum_s cV^(s)[aV^(s)_t]   (fp32 sums in stage order, never written to memory),
//     k_t = khat_t                               keys stored after the rotary embedding (rope_theta == 0), or
//     k_t = RoPE(khat_t, t)                      keys quantised before it (rotate-half convention, angle = t theta^(-2i/hd)).
// Without RoPE the keys are never even dequantised: q_h . khat_t = sum_s sum_m (q_h[m] . cK^(s)_k[.])[k = aK^(s)_{t,m}], so one table
// QT[s][k][m][h] of S x 256 x 8 x n_rep dot products per (sequence, KV head) turns a token's logit into S x 8 shared-memory
// lookups (one 16-byte entry = the 4 heads; lane l reads sub-vector (l + j) % 8 at step j, so the 8 lanes of a quarter-warp hit
// 8 different bank groups whatever the codes are).  With RoPE the two sub-vectors of a rotary pair (elements i and i + 64) are dequantised in registers,
// rotated with cos / sin((base + off) theta_i) = angle addition of a base per 64 tokens (double precision) and a per-CTA offset
// table, and multiplied with q (held in registers: a thread owns four rotary pairs of every 16th token).  Values: warp = token,
// lane = four output elements; the token's probabilities of all heads are one float4 broadcast from shared memory; with two
// stages the two stage tables are interleaved (codeword k of stage s at row 2 k + s) and the odd sub-vectors' lanes read stage 1
// first, so that the two rows a quarter-warp reads per instruction lie in opposite bank halves.
// Split-K over the tokens (flash-decoding): CTA (split, g, b) keeps a running max / sum per head, k_attn_combine merges the
// splits in split order.  d = 16, hd = 128, K <= 256, up to 4 stages each; fp32 arithmetic, no atomics (bit-reproducible).
#pragma once
#include "gsrq_common.cuh"

namespace gsrq {
namespace attn {

constexpr int kHd = 128, kD = 16, kM = 8, kThreads = 256;
constexpr int kPartStride = kHd + 2;   // m, l, acc[128]

struct AttnParams {
  const float *q;             // [B][Hq][128] fp32 (already rotated when rope_theta > 0)
  const uint8_t *kc, *vc;     // code planes: stage s, head g, row t*8 + m at codes[(s*G + g)*plane_rows + t*8 + m]
  const float *k_shapes, *k_gains, *v_shapes, *v_gains;   // [G][S][K][16], [G][S][K]
  int kS, kK, vS, vK;         // codebook dimensions (S = stages in the arrays)
  int k_stages, v_stages;     // stages used
  long long plane_rows;
  const long long *seq_start, *seq_len;   // [B] first token / number of tokens of each sequence in the planes
  int B, Hq, G, n_rep, n_split;
  float scale, rope_theta;
  float *part;                // [B][G][n_split][n_rep][130]
  float *out;                 // [B][Hq][128]
};

__host__ __device__ inline size_t attn_smem_bytes(int k_stages, int v_stages, int n_rep, bool rope) {
  const int ch = rope ? 256 : 512;
  size_t b = (size_t)v_stages * 256 * kD * 4;                                 // value codeword table
  b += rope ? ((size_t)k_stages * 256 * kD * 4 + 64 * 64 * 8 + 4 * 64 * 8)    // key table, offset / base rotations
            : (size_t)((n_rep + 3) & ~3) * k_stages * kM * 256 * 4;           // q . codeword tables (heads innermost, padded to 4)
  const int hp = (n_rep + 3) & ~3;
  b += (size_t)(hp * ch > n_rep * kHd ? hp * ch : n_rep * kHd) * 4;           // logits / probabilities of the chunk [token][head], first the staged q
  b += (size_t)ch * kM * (size_t)(v_stages == 3 ? 4 : v_stages);              // the chunk's value codes [token][m][stage]
  if (rope) b += (size_t)ch * kM * (size_t)k_stages;                          // and key codes [stage][token][m]
  b += 3 * 8 * 4 + 16;                                                        // running max, sum, rescale per head
  return (b + 15) & ~(size_t)15;
}

// NREP / NS > 0: query heads per KV head and stages (keys = values) fixed at compile time, every loop over them unrolled;
// NREP == 0 && NS == 0: the generic kernel (any n_rep <= 8, 1..4 stages each).
template <bool ROPE, int NREP, int NS>
__device__ __forceinline__ void attn_decode_body(const AttnParams &p) {
  extern __shared__ __align__(16) uint8_t asm_raw[];
  constexpr int CH = ROPE ? 256 : 512;
  constexpr int HMAX = NREP > 0 ? NREP : 8;
  const int sp = blockIdx.x, g = blockIdx.y, b = blockIdx.z, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_rep = NREP > 0 ? NREP : p.n_rep, SK = NS > 0 ? NS : p.k_stages, SV = NS > 0 ? NS : p.v_stages;
  float *vtab = reinterpret_cast<float *>(asm_raw);
  float *ktab = vtab + SV * 256 * kD;                                   // ROPE: key table; else the q . codeword tables
  float2 *cs_off = reinterpret_cast<float2 *>(ktab + SK * 256 * kD);    // ROPE only: [64 offsets][64 frequencies]
  float2 *cs_base = cs_off + 64 * 64;                                   // [4 sub-chunks of 64 tokens][64]
  const int HP = (n_rep + 3) & ~3;                                      // heads padded to a multiple of 4
  float *qt = ktab;                                                     // [SK][256][8][HP]
  float *lg = ROPE ? reinterpret_cast<float *>(cs_base + 4 * 64) : qt + HP * SK * kM * 256;
  const int SVP = SV == 3 ? 4 : SV;                                     // stages of one (token, m) side by side, padded to 1 / 2 / 4 bytes
  uint8_t *vcodes = reinterpret_cast<uint8_t *>(lg + (HP * CH > n_rep * kHd ? HP * CH : n_rep * kHd));   // [CH][8][SVP]
  uint2 *kcodes = reinterpret_cast<uint2 *>(vcodes + ((CH * kM * SVP + 15) & ~15));   // ROPE only: [SK][CH]
  float *m_run = reinterpret_cast<float *>(reinterpret_cast<uint8_t *>(kcodes) + (ROPE ? CH * kM * SK : 0));
  float *l_run = m_run + 8, *sc_h = l_run + 8;

  const long long t_seq0 = p.seq_start[b];
  long long len = p.seq_len[b];
  if (t_seq0 < 0 || len < 0 || t_seq0 + len > p.plane_rows / kM) len = 0;   // a sequence that leaves the code planes is served as empty (zeros), never read
  long long per = (len + p.n_split - 1) / p.n_split;
  per = (per + CH - 1) / CH * CH;
  const long long tb = (long long)sp * per, te = min(len, tb + per);
  const float *qg = p.q + ((long long)b * p.Hq + (long long)g * n_rep) * kHd;

  // ---- tables ----
#pragma unroll 8
  for (int e = tid; e < SV * 256 * kD; e += kThreads) {
    const int s = e / (256 * kD), r = e - s * 256 * kD, k = r >> 4;
    const long long cb = ((long long)g * p.vS + s) * p.vK + k;
    // two stages: codeword k of stage s at float (2 k + s) 16, so that a stage-0 row and a stage-1 row never share a bank
    vtab[NS == 2 ? ((2 * k + s) * kD + (r & 15)) : e] = (k < p.vK) ? __fmul_rn(p.v_gains[cb], p.v_shapes[cb * kD + (r & 15)]) : 0.0f;
  }
  if (ROPE) {
#pragma unroll 8
    for (int e = tid; e < SK * 256 * kD; e += kThreads) {
      const int s = e / (256 * kD), r = e - s * 256 * kD, k = r >> 4;
      const long long cb = ((long long)g * p.kS + s) * p.kK + k;
      ktab[NS == 2 ? ((2 * k + s) * kD + (r & 15)) : e] = (k < p.kK) ? __fmul_rn(p.k_gains[cb], p.k_shapes[cb * kD + (r & 15)]) : 0.0f;   // two stages: as the value table
    }
    for (int e = tid; e < 64 * 64; e += kThreads) {   // rotation by (offset within the chunk) x theta_i, in double
      const int off = e >> 6, i = e & 63;
      double sn, cs;
      sincos((double)off * pow((double)p.rope_theta, -(double)i / 64.0), &sn, &cs);
      cs_off[e] = make_float2((float)cs, (float)sn);
    }
  } else {
    // QT[s][k][m][h] = sum_j q_h[16 m + j] cK^(s)_k[j]; q staged in the (still unused) logits buffer
    for (int e = tid; e < n_rep * kHd; e += kThreads) lg[e] = qg[e];
    __syncthreads();
    // thread per (codeword, sub-vector): consecutive lanes write consecutive entries; a thread's sub-vector m = tid % 8 is the same
    // for all its entries, so its q elements stay in registers (up to 4 heads)
    constexpr bool QREG = HMAX <= 4;
    float qr[QREG ? HMAX : 1][kD];
    if (QREG)
#pragma unroll
      for (int h = 0; h < HMAX; ++h)
#pragma unroll
        for (int j = 0; j < kD; ++j) qr[QREG ? h : 0][j] = (h < n_rep) ? lg[h * kHd + (tid & 7) * kD + j] : 0.0f;
    for (int e = tid; e < SK * 256 * kM; e += kThreads) {
      const int m = e & 7, k = (e >> 3) & 255, s = e >> 11;
      float c[kD];
      const long long cb = ((long long)g * p.kS + s) * p.kK + k;
      const float gk = (k < p.kK) ? p.k_gains[cb] : 0.0f;
#pragma unroll
      for (int j4 = 0; j4 < kD / 4; ++j4) {
        const float4 v = (k < p.kK) ? *reinterpret_cast<const float4 *>(p.k_shapes + cb * kD + 4 * j4) : make_float4(0.f, 0.f, 0.f, 0.f);
        c[4 * j4] = __fmul_rn(gk, v.x); c[4 * j4 + 1] = __fmul_rn(gk, v.y); c[4 * j4 + 2] = __fmul_rn(gk, v.z); c[4 * j4 + 3] = __fmul_rn(gk, v.w);
      }
      float a[(HMAX + 3) & ~3];
#pragma unroll
      for (int h = 0; h < ((HMAX + 3) & ~3); ++h) {
        a[h] = 0.0f;
        if (h < HMAX && h < n_rep)
#pragma unroll
          for (int j = 0; j < kD; ++j) a[h] = fmaf(QREG ? qr[QREG ? h : 0][j] : lg[h * kHd + m * kD + j], c[j], a[h]);
      }
#pragma unroll
      for (int h4 = 0; h4 < (HMAX + 3) / 4; ++h4)
        if (4 * h4 < HP) *reinterpret_cast<float4 *>(qt + (long long)e * HP + 4 * h4) = make_float4(a[4 * h4], a[4 * h4 + 1], a[4 * h4 + 2], a[4 * h4 + 3]);
    }
  }
  float qa[ROPE ? HMAX : 1][4], qb[ROPE ? HMAX : 1][4];   // ROPE: this thread's q elements (pairs i, i + 64) of every head
  if (ROPE) {
    const int i0 = ((tid & 15) >> 2) * kD + (tid & 3) * 4;
#pragma unroll
    for (int h = 0; h < HMAX; ++h)
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        qa[ROPE ? h : 0][e] = (h < n_rep) ? qg[h * kHd + i0 + e] : 0.0f;
        qb[ROPE ? h : 0][e] = (h < n_rep) ? qg[h * kHd + 64 + i0 + e] : 0.0f;
      }
  }
  if (tid < 8) { m_run[tid] = -INFINITY; l_run[tid] = 0.0f; sc_h[tid] = 0.0f; }
  // values: warp w takes the tokens t = w (mod 8) of a chunk, lane l the output elements 4 l .. 4 l + 3 of vhat_t (sum of the stages
  // in registers).  Two stages: the tables are interleaved (codeword k of stage s at row 2 k + s: stage 0 in the lower, stage 1 in
  // the upper bank half) and the lanes of the odd sub-vectors read stage 1 first, so that the two rows a quarter-warp reads per
  // instruction never share a bank; a two-term fp32 sum does not depend on the order, so vhat_t is still the stage-order sum.
  float acc[HMAX][4];
#pragma unroll
  for (int h = 0; h < HMAX; ++h) { acc[h][0] = 0.0f; acc[h][1] = 0.0f; acc[h][2] = 0.0f; acc[h][3] = 0.0f; }
  const int m_out = lane >> 2, j_out = (lane & 3) * 4;
  __syncthreads();

  // Code bytes of this thread's tokens (tid, tid + 256, ...) of a chunk, every stage: fetched one chunk ahead, so that the
  // loads of chunk n + 1 are in flight while chunk n is computed.
  constexpr int TPT = CH / kThreads, SMAX = NS > 0 ? NS : 4;
  uint2 nk[TPT][SMAX], nvc[TPT][SMAX];
  auto fetch = [&](long long t0c) {
#pragma unroll
    for (int i = 0; i < TPT; ++i) {
      const long long t = t0c + tid + i * kThreads;
#pragma unroll
      for (int s = 0; s < SMAX; ++s) {
        nk[i][s] = make_uint2(0u, 0u); nvc[i][s] = make_uint2(0u, 0u);
        if (t < te && s < SK) nk[i][s] = *reinterpret_cast<const uint2 *>(p.kc + ((long long)s * p.G + g) * p.plane_rows + (t_seq0 + t) * kM);
        if (t < te && s < SV) nvc[i][s] = *reinterpret_cast<const uint2 *>(p.vc + ((long long)s * p.G + g) * p.plane_rows + (t_seq0 + t) * kM);
      }
    }
  };
  fetch(tb);

  for (long long t0 = tb; t0 < te; t0 += CH) {
    const int nv = (int)min((long long)CH, te - t0);   // valid tokens of the chunk
    // the chunk's value codes -> shared memory, the stages of one sub-vector side by side; key codes: shared memory (RoPE: any
    // thread needs any token) or this thread's registers
    uint2 ck[TPT][SMAX];
#pragma unroll
    for (int i = 0; i < TPT; ++i) {
      const int t = tid + i * kThreads;
      if (NS == 2) {
        const uint2 a = nvc[i][0], c = nvc[i][1];
        reinterpret_cast<uint4 *>(vcodes)[t] = make_uint4(__byte_perm(a.x, c.x, 0x5140), __byte_perm(a.x, c.x, 0x7362),
                                                          __byte_perm(a.y, c.y, 0x5140), __byte_perm(a.y, c.y, 0x7362));
      } else {
#pragma unroll
        for (int s = 0; s < SMAX; ++s) {
          if (s >= SV) break;
          const uint2 v = nvc[i][s];
          if (SVP == 1) reinterpret_cast<uint2 *>(vcodes)[t] = v;
          else
#pragma unroll
            for (int m = 0; m < kM; ++m) vcodes[(t * kM + m) * SVP + s] = (uint8_t)(((m < 4 ? v.x : v.y) >> (8 * (m & 3))) & 255u);
        }
      }
#pragma unroll
      for (int s = 0; s < SMAX; ++s) {
        ck[i][s] = nk[i][s];
        if (ROPE && s < SK) kcodes[s * CH + t] = nk[i][s];
      }
    }
    if (t0 + CH < te) fetch(t0 + CH);
    // ---- logits ----
    if (!ROPE) {
#pragma unroll
      for (int i = 0; i < TPT; ++i) {
        const int t = tid + i * kThreads;
        if (t >= nv) break;
        float sum[(HMAX + 3) & ~3];
#pragma unroll
        for (int h = 0; h < ((HMAX + 3) & ~3); ++h) sum[h] = 0.0f;
#pragma unroll
        for (int s = 0; s < (NS > 0 ? NS : 4); ++s) {
          if (s >= SK) break;
          const uint2 cw = ck[i][s];
#pragma unroll
          for (int j = 0; j < kM; ++j) {
            // lane l takes sub-vector (l + j) % 8 at step j: the eight lanes of a quarter-warp read eight different sub-vectors'
            // entries, which the table layout puts in eight different 16-byte bank groups (no conflicts whatever the codes are)
            const int m = (lane + j) & 7;
            const int k = (int)(__byte_perm(cw.x, cw.y, m) & 255u);
            const float4 *q4 = reinterpret_cast<const float4 *>(qt + ((s * 256 + k) * kM + m) * HP);
#pragma unroll
            for (int h4 = 0; h4 < (HMAX + 3) / 4; ++h4) {
              if (4 * h4 >= n_rep) break;
              const float4 v = q4[h4];
              sum[4 * h4] += v.x;
              if (4 * h4 + 1 < HMAX) sum[4 * h4 + 1] += v.y;
              if (4 * h4 + 2 < HMAX) sum[4 * h4 + 2] += v.z;
              if (4 * h4 + 3 < HMAX) sum[4 * h4 + 3] += v.w;
            }
          }
        }
#pragma unroll
        for (int h4 = 0; h4 < (HMAX + 3) / 4; ++h4)
          if (4 * h4 < n_rep)
            *reinterpret_cast<float4 *>(lg + t * HP + 4 * h4) =
                make_float4(sum[4 * h4] * p.scale, sum[4 * h4 + 1] * p.scale, sum[4 * h4 + 2] * p.scale, sum[4 * h4 + 3] * p.scale);
      }
    } else {
      // Thread = (token slot tid / 16, rotary sub-vector pair mq, quad jq): the pairs i = 16 mq + 4 jq + e and i + 64, e < 4, of the
      // tokens slot, slot + 16, ... of each 64-token sub-chunk; its 8 q elements per head stay in registers for the whole CTA.
      {   // rotation by (first position of each sub-chunk) x theta_i, in double
        const int sub = tid >> 6, i = tid & 63;
        double sn, cs;
        sincos((double)(t0 + 64 * sub) * pow((double)p.rope_theta, -(double)i / 64.0), &sn, &cs);
        cs_base[tid] = make_float2((float)cs, (float)sn);
      }
      __syncthreads();
      const int l16 = tid & 15, slot = tid >> 4, mq = l16 >> 2, i0 = mq * kD + (l16 & 3) * 4;
#pragma unroll 1
      for (int sub = 0; sub < CH / 64; ++sub) {
        if (sub * 64 >= nv) break;
        float2 cb[4];
        {
          const float4 b0 = *reinterpret_cast<const float4 *>(cs_base + sub * 64 + i0), b1 = *reinterpret_cast<const float4 *>(cs_base + sub * 64 + i0 + 2);
          cb[0] = make_float2(b0.x, b0.y); cb[1] = make_float2(b0.z, b0.w); cb[2] = make_float2(b1.x, b1.y); cb[3] = make_float2(b1.z, b1.w);
        }
#pragma unroll
        for (int it = 0; it < 4; ++it) {
          const int off = it * 16 + slot, t = sub * 64 + off;
          const bool ok = t < nv;
          float a[4] = {0.f, 0.f, 0.f, 0.f}, bb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int st = 0; st < (NS > 0 ? NS : 4); ++st) {
            if (st >= SK) break;
            // two stages: the odd sub-vector pairs take stage 1 first, so that the two rows a quarter-warp reads per instruction lie in
            // opposite bank halves (a two-term fp32 sum does not depend on the order)
            const int s = (NS == 2) ? (st ^ (mq & 1)) : st;
            const uint2 cw = kcodes[s * CH + t];
            const int ra = (NS == 2) ? (2 * ((cw.x >> (8 * mq)) & 255u) + s) : (s * 256 + ((cw.x >> (8 * mq)) & 255u));
            const int rb = (NS == 2) ? (2 * ((cw.y >> (8 * mq)) & 255u) + s) : (s * 256 + ((cw.y >> (8 * mq)) & 255u));
            const float4 va = *reinterpret_cast<const float4 *>(ktab + ra * kD + (l16 & 3) * 4);
            const float4 vb = *reinterpret_cast<const float4 *>(ktab + rb * kD + (l16 & 3) * 4);
            if (st == 0) { a[0] = va.x; a[1] = va.y; a[2] = va.z; a[3] = va.w; bb[0] = vb.x; bb[1] = vb.y; bb[2] = vb.z; bb[3] = vb.w; }
            else { a[0] = __fadd_rn(a[0], va.x); a[1] = __fadd_rn(a[1], va.y); a[2] = __fadd_rn(a[2], va.z); a[3] = __fadd_rn(a[3], va.w);
                   bb[0] = __fadd_rn(bb[0], vb.x); bb[1] = __fadd_rn(bb[1], vb.y); bb[2] = __fadd_rn(bb[2], vb.z); bb[3] = __fadd_rn(bb[3], vb.w); }
          }
          float2 co[4];
          {
            // this lane's 32 bytes in two loads, the halves in the order that gives the eight lanes of a quarter-warp eight different bank groups
            const int sw = ((l16 & 3) + mq) & 1;
            const float4 f0 = *reinterpret_cast<const float4 *>(cs_off + off * 64 + i0 + 2 * sw), f1 = *reinterpret_cast<const float4 *>(cs_off + off * 64 + i0 + 2 * (1 - sw));
            const float4 o0 = sw ? f1 : f0, o1 = sw ? f0 : f1;
            co[0] = make_float2(o0.x, o0.y); co[1] = make_float2(o0.z, o0.w); co[2] = make_float2(o1.x, o1.y); co[3] = make_float2(o1.z, o1.w);
          }
          float part[HMAX];
#pragma unroll
          for (int h = 0; h < HMAX; ++h) part[h] = 0.0f;
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float c = cb[e].x * co[e].x - cb[e].y * co[e].y, sn = cb[e].y * co[e].x + cb[e].x * co[e].y;
            const float ar = a[e] * c - bb[e] * sn, br = bb[e] * c + a[e] * sn;
#pragma unroll
            for (int h = 0; h < HMAX; ++h)
              if (h < n_rep) part[h] = fmaf(qa[h][e], ar, fmaf(qb[h][e], br, part[h]));
          }
          // sum over the token's 16 threads
          if (HMAX == 4) {   // 4 heads: exchange halves first (5 shuffles instead of 16); lane l16 < 4 ends with head 2 (l16 & 1) + (l16 >> 1)
            const bool b0 = l16 & 1, b1 = l16 & 2;
            float v0 = (b0 ? part[2] : part[0]) + __shfl_xor_sync(0xffffffffu, b0 ? part[0] : part[2], 1);
            float v1 = (b0 ? part[3] : part[1]) + __shfl_xor_sync(0xffffffffu, b0 ? part[1] : part[3], 1);
            float r = (b1 ? v1 : v0) + __shfl_xor_sync(0xffffffffu, b1 ? v0 : v1, 2);
            r += __shfl_xor_sync(0xffffffffu, r, 4);
            r += __shfl_xor_sync(0xffffffffu, r, 8);
            if (l16 < 4 && ok) lg[t * HP + 2 * (l16 & 1) + (l16 >> 1)] = r * p.scale;
          } else {
#pragma unroll
            for (int h = 0; h < HMAX; ++h) {
              if (h < n_rep) {
                float v = part[h];
                v += __shfl_xor_sync(0xffffffffu, v, 1);
                v += __shfl_xor_sync(0xffffffffu, v, 2);
                v += __shfl_xor_sync(0xffffffffu, v, 4);
                v += __shfl_xor_sync(0xffffffffu, v, 8);
                if (l16 == 0 && ok) lg[t * HP + h] = v * p.scale;
              }
            }
          }
        }
      }
    }
    __syncthreads();
    // ---- running softmax: warp h handles head h ----
    if (warp < n_rep) {
      const int h = warp;
      float mx = -INFINITY;
      for (int t = lane; t < nv; t += 32) mx = fmaxf(mx, lg[t * HP + h]);
      for (int off = 16; off; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, off));
      const float m_old = m_run[h], m_new = fmaxf(m_old, mx);
      float sum = 0.0f;
      for (int t = lane; t < CH; t += 32) {
        const float pr = (t < nv) ? expf(lg[t * HP + h] - m_new) : 0.0f;
        lg[t * HP + h] = pr;
        sum += pr;
      }
      for (int off = 16; off; off >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, off);
      if (lane == 0) {
        const float sc = (m_old == -INFINITY) ? 0.0f : expf(m_old - m_new);
        sc_h[h] = sc;
        l_run[h] = l_run[h] * sc + sum;
        m_run[h] = m_new;
      }
    }
    __syncthreads();
    // ---- values: warp = token (t = warp, warp + 8, ...), lane = output elements 4 lane .. 4 lane + 3 ----
#pragma unroll
    for (int h = 0; h < HMAX; ++h)
      if (h < n_rep) {
        const float sc = sc_h[h];
        acc[h][0] *= sc; acc[h][1] *= sc; acc[h][2] *= sc; acc[h][3] *= sc;
      }
    auto value_of = [&](int t) -> float4 {   // vhat_t[4 lane .. 4 lane + 3] = sum over the stages, fp32, stage order
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      const uint8_t *cp = vcodes + (t * kM + m_out) * SVP;
      unsigned cw;                            // the stages' code bytes of this lane's sub-vector, one load
      if (NS == 1) cw = *cp;
      else if (NS == 2) cw = *reinterpret_cast<const unsigned short *>(cp);
      else if (SVP == 4) cw = *reinterpret_cast<const unsigned *>(cp);
      else if (SVP == 2) cw = *reinterpret_cast<const unsigned short *>(cp);
      else cw = *cp;
      if (NS == 2) {
        const int s1 = m_out & 1;   // stage read first
        const float4 ca = *reinterpret_cast<const float4 *>(vtab + (2 * ((cw >> (8 * s1)) & 255u) + s1) * kD + j_out);
        const float4 cb = *reinterpret_cast<const float4 *>(vtab + (2 * ((cw >> (8 * (1 - s1))) & 255u) + (1 - s1)) * kD + j_out);
        return make_float4(__fadd_rn(ca.x, cb.x), __fadd_rn(ca.y, cb.y), __fadd_rn(ca.z, cb.z), __fadd_rn(ca.w, cb.w));
      }
#pragma unroll
      for (int s = 0; s < (NS > 0 ? NS : 4); ++s) {
        if (s >= SV) break;
        const float4 c = *reinterpret_cast<const float4 *>(vtab + (s * 256 + ((cw >> (8 * s)) & 255u)) * kD + j_out);
        if (s == 0) v = c;
        else { v.x = __fadd_rn(v.x, c.x); v.y = __fadd_rn(v.y, c.y); v.z = __fadd_rn(v.z, c.z); v.w = __fadd_rn(v.w, c.w); }
      }
      return v;
    };
    auto add_token = [&](int t, const float4 &v) {   // acc_h += p_h(t) vhat_t: the token's probabilities as float4 broadcasts
#pragma unroll
      for (int h4 = 0; h4 < (HMAX + 3) / 4; ++h4) {
        if (4 * h4 >= n_rep) break;
        const float4 pr = *reinterpret_cast<const float4 *>(lg + t * HP + 4 * h4);
        const float pv[4] = {pr.x, pr.y, pr.z, pr.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int h = 4 * h4 + i;
          if (h < HMAX && h < n_rep) {
            acc[h][0] = fmaf(pv[i], v.x, acc[h][0]); acc[h][1] = fmaf(pv[i], v.y, acc[h][1]);
            acc[h][2] = fmaf(pv[i], v.z, acc[h][2]); acc[h][3] = fmaf(pv[i], v.w, acc[h][3]);
          }
        }
      }
    };
    int t = warp;
    for (; t + 24 < nv; t += 32) {   // four tokens in flight
      const float4 v0 = value_of(t), v1 = value_of(t + 8), v2 = value_of(t + 16), v3 = value_of(t + 24);
      add_token(t, v0);
      add_token(t + 8, v1);
      add_token(t + 16, v2);
      add_token(t + 24, v3);
    }
    for (; t < nv; t += 8) add_token(t, value_of(t));
    __syncthreads();
  }
  // ---- this split's result: m, l, acc = the eight warps' partial sums added in warp order ----
  float *ex = reinterpret_cast<float *>(asm_raw);   // [8 warps][n_rep][128]: the codeword tables are no longer needed
  float *pp = p.part + (((long long)b * p.G + g) * p.n_split + sp) * n_rep * kPartStride;
#pragma unroll
  for (int h = 0; h < HMAX; ++h)
    if (h < n_rep) {
      *reinterpret_cast<float4 *>(ex + ((warp * n_rep + h) * kHd) + 4 * lane) = make_float4(acc[h][0], acc[h][1], acc[h][2], acc[h][3]);
    }
  __syncthreads();
  for (int e = tid; e < n_rep * kHd; e += kThreads) {
    float sum = 0.0f;
#pragma unroll
    for (int w8 = 0; w8 < 8; ++w8) sum += ex[w8 * n_rep * kHd + e];
    pp[(e >> 7) * kPartStride + 2 + (e & 127)] = sum;
  }
  if (tid < n_rep) { pp[tid * kPartStride] = m_run[tid]; pp[tid * kPartStride + 1] = l_run[tid]; }
}

// Two entry points so that the register budgets differ: the RoPE body is held to 128 registers (two CTAs per SM, which shared
// memory allows), the table-lookup body is left to the compiler (about 100).
template <bool ROPE, int NREP, int NS>
__global__ void __launch_bounds__(kThreads) k_attn_decode(AttnParams p) { attn_decode_body<ROPE, NREP, NS>(p); }
template <int NREP, int NS>
__global__ void __launch_bounds__(kThreads, 2) k_attn_decode_rope(AttnParams p) { attn_decode_body<true, NREP, NS>(p); }

// ---- the paper's own operating point: d = head_dim = 128 (one sub-vector per token and head), up to 32 stages ----
// The codeword tables of that point (stages x 256 x 128 fp32 = 1.5 MB per head at R = 12) do not fit in shared memory, so this
// kernel dequantises from the codebooks as they lie in global memory (L2-resident: every CTA of a KV head reads the same rows):
// a warp owns every 8th token of the split; lane l holds channels 4l .. 4l + 3 of khat_t and vhat_t (fp32 sums in stage order,
// c = fl32(g_k s_k), exactly gsrq_decode's), rotates the key when rope_theta > 0 (pair (i, i + 64): lanes l and l ^ 16; angle in
// double), reduces the n_rep logits over the warp and keeps a running max / sum / accumulator per query head.  The 8 warps are
// merged in warp order into the same partial record the d = 16 kernels write (k_attn_combine merges the splits).  No atomics.
// Functional first: per token it reads 2 x stages x 512 bytes of codeword rows from L2, which bounds it far below the HBM rate
// of the codes.  grid = (n_split, G, B), block = 256, static shared memory only.
template <bool ROPE>
__global__ void __launch_bounds__(kThreads, 2) k_attn_decode_wide(AttnParams p) {
  __shared__ float sm_m[8][8], sm_l[8][8];
  __shared__ __align__(16) float sm_acc[8][8][kHd];   // [warp][head][channel]
  const int sp = blockIdx.x, g = blockIdx.y, b = blockIdx.z, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_rep = p.n_rep;
  const long long t_seq0 = p.seq_start[b];
  long long len = p.seq_len[b];
  if (t_seq0 < 0 || len < 0 || t_seq0 + len > p.plane_rows) len = 0;   // M = 1: plane_rows is the number of tokens in the planes
  const long long per = (len + p.n_split - 1) / p.n_split;
  const long long tb = (long long)sp * per, te = min(len, tb + per);
  float q[8][4], acc[8][4], m_run[8], l_run[8];
#pragma unroll
  for (int h = 0; h < 8; ++h) {
    const float4 v = (h < n_rep) ? *reinterpret_cast<const float4 *>(p.q + ((long long)b * p.Hq + (long long)g * n_rep + h) * kHd + 4 * lane)
                                 : make_float4(0.f, 0.f, 0.f, 0.f);
    q[h][0] = v.x; q[h][1] = v.y; q[h][2] = v.z; q[h][3] = v.w;
    acc[h][0] = acc[h][1] = acc[h][2] = acc[h][3] = 0.0f;
    m_run[h] = -INFINITY; l_run[h] = 0.0f;
  }
  double inv_freq[4] = {0.0, 0.0, 0.0, 0.0};
  if (ROPE)
#pragma unroll
    for (int j = 0; j < 4; ++j) inv_freq[j] = pow((double)p.rope_theta, -(double)(4 * (lane & 15) + j) / 64.0);
  const float *ksh = p.k_shapes + (long long)g * p.kS * p.kK * kHd, *kga = p.k_gains + (long long)g * p.kS * p.kK;
  const float *vsh = p.v_shapes + (long long)g * p.vS * p.vK * kHd, *vga = p.v_gains + (long long)g * p.vS * p.vK;
  // xhat = ((c_0 + c_1) + ...) in fp32, stage order; four stages' gain and row loads are issued together (latency), then added in order
  auto dequant = [&](int code_l, int ns, const float *sh, const float *ga, int Kc, float (&x)[4]) {
    for (int s0 = 0; s0 < ns; s0 += 4) {
      float gk[4];
      float4 sv[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int s = min(s0 + u, ns - 1);   // past the last stage: a valid (repeated) load that is not added
        const long long cbi = (long long)s * Kc + __shfl_sync(0xffffffffu, code_l, s);
        gk[u] = __ldg(ga + cbi);
        sv[u] = __ldg(reinterpret_cast<const float4 *>(sh + cbi * kHd) + lane);
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (s0 + u >= ns) break;
        const float c0 = __fmul_rn(gk[u], sv[u].x), c1 = __fmul_rn(gk[u], sv[u].y), c2 = __fmul_rn(gk[u], sv[u].z), c3 = __fmul_rn(gk[u], sv[u].w);
        if (s0 + u == 0) { x[0] = c0; x[1] = c1; x[2] = c2; x[3] = c3; }
        else { x[0] = __fadd_rn(x[0], c0); x[1] = __fadd_rn(x[1], c1); x[2] = __fadd_rn(x[2], c2); x[3] = __fadd_rn(x[3], c3); }
      }
    }
  };
  for (long long t = tb + warp; t < te; t += 8) {
    // lane s holds the code byte of stage s (keys and values)
    const long long tok = t_seq0 + t;
    const int kcode = (lane < p.k_stages) ? min((int)p.kc[((long long)lane * p.G + g) * p.plane_rows + tok], p.kK - 1) : 0;
    const int vcode = (lane < p.v_stages) ? min((int)p.vc[((long long)lane * p.G + g) * p.plane_rows + tok], p.vK - 1) : 0;
    float kh[4], vh[4];
    dequant(kcode, p.k_stages, ksh, kga, p.kK, kh);
    dequant(vcode, p.v_stages, vsh, vga, p.vK, vh);
    if (ROPE) {   // rotate-half: (a, b) = (x_i, x_{i + 64}) -> (a cos - b sin, b cos + a sin), angle = t * theta^(-2 i / 128)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        double sn, cs;
        sincos((double)t * inv_freq[j], &sn, &cs);
        const float mine = kh[j], other = __shfl_xor_sync(0xffffffffu, mine, 16);
        kh[j] = (lane < 16) ? fmaf(mine, (float)cs, -other * (float)sn) : fmaf(mine, (float)cs, other * (float)sn);
      }
    }
#pragma unroll
    for (int h = 0; h < 8; ++h) {
      if (h >= n_rep) break;
      float dot = fmaf(q[h][0], kh[0], fmaf(q[h][1], kh[1], fmaf(q[h][2], kh[2], q[h][3] * kh[3])));
#pragma unroll
      for (int off = 16; off; off >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, off);
      const float lg = dot * p.scale;
      const float m_new = fmaxf(m_run[h], lg);
      const float resc = (m_run[h] == -INFINITY) ? 0.0f : expf(m_run[h] - m_new);
      const float pr = expf(lg - m_new);
      l_run[h] = fmaf(l_run[h], resc, pr);
#pragma unroll
      for (int j = 0; j < 4; ++j) acc[h][j] = fmaf(acc[h][j], resc, pr * vh[j]);
      m_run[h] = m_new;
    }
  }
  // ---- the split's record: the eight warps merged in warp order ----
#pragma unroll
  for (int h = 0; h < 8; ++h) {
    if (h >= n_rep) break;
    if (lane == 0) { sm_m[warp][h] = m_run[h]; sm_l[warp][h] = l_run[h]; }
    *reinterpret_cast<float4 *>(&sm_acc[warp][h][4 * lane]) = make_float4(acc[h][0], acc[h][1], acc[h][2], acc[h][3]);
  }
  __syncthreads();
  float *pp = p.part + (((long long)b * p.G + g) * p.n_split + sp) * n_rep * kPartStride;
  for (int e = tid; e < n_rep * kHd; e += kThreads) {
    const int h = e >> 7, c = e & 127;
    float M = -INFINITY;
#pragma unroll
    for (int w8 = 0; w8 < 8; ++w8) M = fmaxf(M, sm_m[w8][h]);
    float L = 0.0f, o = 0.0f;
#pragma unroll
    for (int w8 = 0; w8 < 8; ++w8) {
      const float wgt = (sm_m[w8][h] == -INFINITY) ? 0.0f : expf(sm_m[w8][h] - M);
      L = fmaf(sm_l[w8][h], wgt, L);
      o = fmaf(sm_acc[w8][h][c], wgt, o);
    }
    pp[h * kPartStride + 2 + c] = o;
    if (c == 0) { pp[h * kPartStride] = M; pp[h * kPartStride + 1] = L; }
  }
}

// Merge the splits of one (sequence, query head) in split order.  grid = (Hq, B), block = 128.
__global__ void __launch_bounds__(128) k_attn_combine(AttnParams p) {
  const int hq = blockIdx.x, b = blockIdx.y, e = threadIdx.x;
  const int g = hq / p.n_rep, h = hq - g * p.n_rep;
  const float *pp = p.part + (((long long)b * p.G + g) * p.n_split) * p.n_rep * kPartStride + h * kPartStride;
  const long long st = (long long)p.n_rep * kPartStride;
  float M = -INFINITY;
  for (int s = 0; s < p.n_split; ++s) M = fmaxf(M, pp[s * st]);
  float L = 0.0f, o = 0.0f;
  for (int s = 0; s < p.n_split; ++s) {
    const float ms = pp[s * st];
    const float w = (ms == -INFINITY) ? 0.0f : expf(ms - M);
    L += pp[s * st + 1] * w;
    o += pp[s * st + 2 + e] * w;
  }
  p.out[((long long)b * p.Hq + hq) * kHd + e] = (L > 0.0f) ? o / L : 0.0f;
}

}  // namespace attn
}  // namespace gsrq
