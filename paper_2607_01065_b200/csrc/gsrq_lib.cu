// gsrq_lib.cu -- host side of libgsrq: argument checks, workspace plan, kernel launches.
// Every step of the path runs in the kernels under csrc/; this file only orchestrates.
#include <stdarg.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <vector>

#include "gsrq_common.cuh"
#include "k_codec.cuh"
#include "k_prep.cuh"
#include "k_update.cuh"
#include "k_score.cuh"
#include "k_score_tc.cuh"
#include "k_fit_tc.cuh"
#include "k_encode_tc.cuh"
#include "k_wide.cuh"
#include "k_score_tc_wide.cuh"
#include "k_attn.cuh"
#include "k_variants.cuh"

namespace gsrq {

static_assert(sizeof(gsrq_view) == 40 && sizeof(gsrq_codebook) == 24 && sizeof(gsrq_fit_stats) == 24 + 16 * GSRQ_MAX_ITERS, "ABI layout");
static thread_local char g_err[512] = "";

void set_error(const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}


// ---- launch accounting / optional per-kernel CUDA-event timing (gsrq_profile_*) ----
enum { kClsPrep = 0, kClsScore = 1, kClsRefine = 2, kClsUpdate = 3, kClsMisc = 4, kClsDecode = 5, kClsEncode = 6, kNumCls = 7 };
struct ProfRec { int cls; cudaEvent_t a, b; };
static std::mutex g_prof_mu;
static std::vector<ProfRec> g_prof_recs;
static bool g_prof_on = false;
static long long g_launches[kNumCls] = {0, 0, 0, 0, 0, 0, 0};

struct ProfScope {
  cudaStream_t stream;
  cudaEvent_t b = nullptr;
  ProfScope(int cls, cudaStream_t s) : stream(s) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    g_launches[cls]++;
    if (g_prof_on) {
      ProfRec r{cls, nullptr, nullptr};
      if (cudaEventCreate(&r.a) == cudaSuccess && cudaEventCreate(&r.b) == cudaSuccess) {
        cudaEventRecord(r.a, stream);
        b = r.b;
        g_prof_recs.push_back(r);
      }
    }
  }
  ~ProfScope() { if (b) cudaEventRecord(b, stream); }
};
#define LAUNCH(cls, stream, ...) do { gsrq::ProfScope _ps(cls, stream); __VA_ARGS__; } while (0)

static inline size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// SM count of the CURRENT device (cached per device ordinal; the cache is only ever written with the same value).
static int sm_count() {
  static int cache[64] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 148;
  if (dev >= 0 && dev < 64 && cache[dev] > 0) return cache[dev];
  int n = 0;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
  if (dev >= 0 && dev < 64) cache[dev] = n;
  return n;
}

struct Plan {
  long long nf_tok, Nf, Nall, nE;
  int M;
  // [0, encode_total): what gsrq_encode needs; the rest is for the fit
  size_t off_list, off_cnt, off_st, off_ebimg, off_egmax, off_eres, encode_total;
  size_t off_Rf, off_coef, off_wt, off_idx, off_ids, off_epart, off_term;
  size_t off_ahi, off_alo, off_rnorm, off_bimg, off_gmax, off_wn, off_part, off_bar, off_clk, off_chg, total;
  long long chg_stride_g;
};

constexpr int kNumCounters = 256;
constexpr int kMaxCtas = 256;  // upper bound of co-resident CTAs (SMs) the partial buffer is sized for
constexpr int kTermStride = GSRQ_MAX_ITERS + 1;

// n_fit_tokens: > 0 fit subset size, 0 = fit on all tokens, < 0 = no fit (encode / decode only)
static Plan make_plan(const gsrq_view *v, int K, int S, long long n_fit_tokens) {
  (void)K;
  Plan p;
  p.M = v->hd / v->d;
  p.nf_tok = (n_fit_tokens > 0) ? n_fit_tokens : (n_fit_tokens == 0 ? v->T : 0);
  p.Nf = p.nf_tok * p.M;
  p.Nall = v->T * p.M;
  p.nE = (p.Nf + kPrepRows - 1) / kPrepRows;
  size_t o = 0;
  p.off_list = o; o += align_up((size_t)v->G * p.Nall * sizeof(uint2));
  p.off_cnt = o;  o += align_up(kNumCounters * sizeof(unsigned int));
  p.off_st = o;   o += align_up((size_t)v->G * sizeof(DevStats));
  p.off_ebimg = o; o += align_up(v->d == tc::kD ? (size_t)v->G * tc::kEncMaxS * 3 * tc::kBImgBytes : 0);
  p.off_egmax = o; o += align_up(v->d == tc::kD ? (size_t)v->G * tc::kEncMaxS * sizeof(int) : 0);
  // fp32 residual between the chained tensor-core passes of an encode with more than kEncMaxS stages
  p.off_eres = o;  o += align_up((v->d == tc::kD && S > tc::kEncMaxS) ? (size_t)v->G * p.Nall * v->d * sizeof(float) : 0);
  p.encode_total = o;
  p.off_Rf = o;   o += align_up((size_t)v->G * p.Nf * v->d * sizeof(float));
  p.off_coef = o; o += align_up((size_t)v->G * p.Nf * 2 * sizeof(double));  // per-row {w, w/(||r||+eps)}
  p.off_wt = o;   o += align_up((size_t)v->G * p.nf_tok * sizeof(float));
  p.off_idx = o;  o += align_up((size_t)v->G * p.Nf);
  p.off_ids = o;  o += align_up((size_t)v->G * GSRQ_MAX_K * sizeof(long long));
  p.off_epart = o; o += align_up((size_t)v->G * p.nE * sizeof(double));
  p.off_term = o; o += align_up(p.Nf ? (size_t)v->G * kTermStride * 256 * sizeof(double) : 0);
  const bool tcp = (v->d == tc::kD);
  p.off_ahi = o;   o += align_up(tcp ? (size_t)v->G * p.Nf * tc::kD * 2 : 0);
  p.off_alo = o;   o += align_up(tcp ? (size_t)v->G * p.Nf * tc::kD * 2 : 0);
  p.off_rnorm = o; o += align_up(tcp ? (size_t)v->G * p.Nf * sizeof(float) : 0);
  p.off_bimg = o;  o += align_up(tcp ? (size_t)v->G * 3 * tc::kBImgBytes : 0);
  p.off_gmax = o;  o += align_up(tcp ? (size_t)v->G * sizeof(int) : 0);
  // fused fit kernel (d == 16): per-row w/(||r||+eps), per-CTA partials [G][nx][256][34] with G * nx <= kMaxCtas, group barriers
  p.off_wn = o;    o += align_up(tcp ? (size_t)v->G * p.Nf * sizeof(double) : 0);
  p.off_part = o;  o += align_up(tcp && p.Nf ? (size_t)(v->G > kMaxCtas ? v->G : kMaxCtas) * tc::kN * tc::kFitP * sizeof(double) : 0);
  p.off_bar = o;   o += align_up(tcp ? (size_t)v->G * sizeof(unsigned int) : 0);
  p.off_clk = o;   o += align_up(tcp ? (size_t)(v->G > kMaxCtas ? v->G : kMaxCtas) * 16 * sizeof(long long) : 0);
  // change lists of the incremental reduction: per group 128 entries per tile + 512 per CTA (k_fit_tc.cuh)
  p.chg_stride_g = ((p.Nf + tc::kTileM - 1) / tc::kTileM) * tc::kTileM + 512LL * kMaxCtas;
  p.off_chg = o;   o += align_up(tcp && p.Nf ? (size_t)v->G * p.chg_stride_g * sizeof(uint2) : 0);
  p.total = o;
  return p;
}

static inline bool is_wide(int d) { return d == 64 || d == 128 || d == 256; }   // the paper's operating points (k_wide.cuh)

static int check_view(const gsrq_view *v, int K, int S) {
  if (!v) { set_error("view is NULL"); return GSRQ_EINVAL; }
  if (v->dtype != GSRQ_F32 && v->dtype != GSRQ_BF16) { set_error("view.dtype must be GSRQ_F32 or GSRQ_BF16"); return GSRQ_EINVAL; }
  if (v->G <= 0 || v->T <= 0 || v->hd <= 0 || v->d <= 0 || v->hd % v->d) { set_error("bad view shape (G=%d T=%lld hd=%d d=%d)", v->G, (long long)v->T, v->hd, v->d); return GSRQ_EINVAL; }
  if (K <= 0 || K > GSRQ_MAX_K) { set_error("K must be in [1, %d], got %d", GSRQ_MAX_K, K); return GSRQ_EINVAL; }
  if (S <= 0 || S > GSRQ_MAX_STAGES) { set_error("S must be in [1, %d], got %d", GSRQ_MAX_STAGES, S); return GSRQ_EINVAL; }
  if (v->d != 8 && v->d != 16 && v->d != 32 && !is_wide(v->d)) { set_error("d = %d: this build has kernels for d in {8, 16, 32, 64, 128, 256}", v->d); return GSRQ_EUNSUPPORTED; }
  const int al = (v->dtype == GSRQ_BF16) ? 8 : 4;  // 16-byte vector loads
  if (v->stride_g % al || v->stride_t % al) { set_error("strides must be multiples of %d elements (16-byte loads)", al); return GSRQ_EINVAL; }
  if ((long long)v->G * v->T * (v->hd / v->d) >= (1LL << 32)) { set_error("G*T*M must be < 2^32"); return GSRQ_EINVAL; }
  return GSRQ_OK;
}

// Tensors are read / written with 16-byte vector accesses: a misaligned base would fault instead of returning an error.
static int check_align16(const void *ptr, const char *what) {
  if (ptr && ((uintptr_t)ptr & 15)) { set_error("%s must be 16-byte aligned", what); return GSRQ_EINVAL; }
  return GSRQ_OK;
}

static int check_ws(const void *ws, size_t bytes, size_t need) {
  if (!ws || ((uintptr_t)ws & 255)) { set_error("workspace must be non-NULL and 256-byte aligned"); return GSRQ_EWORKSPACE; }
  if (bytes < need) { set_error("workspace too small: %zu < %zu bytes", bytes, need); return GSRQ_EWORKSPACE; }
  return GSRQ_OK;
}

static RowSrc make_src(const void *kv, const gsrq_view *v, const float *rows, long long rows_per_group) {
  RowSrc s;
  s.kv = kv; s.rows = rows; s.dtype = v->dtype; s.M = v->hd / v->d; s.d = v->d;
  s.stride_g = v->stride_g; s.stride_t = v->stride_t; s.rows_per_group = rows_per_group;
  return s;
}

#define DISPATCH_D(d, ...)                          \
  do {                                              \
    if ((d) == 8) { constexpr int D = 8; __VA_ARGS__; }   \
    else if ((d) == 16) { constexpr int D = 16; __VA_ARGS__; } \
    else { constexpr int D = 32; __VA_ARGS__; }     \
  } while (0)

static int run_encode_tc(const void *kv, const gsrq_view *v, const float *rows0, long long N, const gsrq_codebook *cb, int n_stages,
                         uint8_t *codes, long long code_stride_s, float *carry, bool want_residual, const struct Plan &pl, char *ws,
                         unsigned int *cnt_base, cudaStream_t stream);
static bool use_tc(int d);

// One filter + refine pass (assignment or multi-stage encode) described by `p`.
static int run_encode(EncParams p, int G, int d, cudaStream_t stream) {
  constexpr int RPT = 2;
  const size_t smem = ((size_t)p.K * d + p.K + 4) * sizeof(float);
  dim3 grid((unsigned)((p.N + 256 * RPT - 1) / (256 * RPT)), (unsigned)G);
  LAUNCH(kClsScore, stream, DISPATCH_D(d, (k_encode<D, RPT><<<grid, 256, smem, stream>>>(p))));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  LAUNCH(kClsRefine, stream, DISPATCH_D(d, (k_encode_exact<D><<<1184, 256, 0, stream>>>(p))));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

// One update (reduction + Eq. 7 / Eq. 8 + operand images) of the stage slice from the assignment `idx`.
static int run_update(const Plan &pl, const gsrq_view *v, int K, char *ws, const uint8_t *idx, float *shapes_st,
                      float *gains_st, long long cb_stride_g, DevStats *st, int lloyd, int t, bool images, cudaStream_t stream) {
  const int d = v->d;
  UpdParams u{};
  u.Rf = (const float *)(ws + pl.off_Rf); u.coef = (const double2 *)(ws + pl.off_coef);
  u.idx = idx; u.Nf = pl.Nf; u.M = pl.M; u.K = K; u.shapes = shapes_st; u.gains = gains_st; u.cb_stride_g = cb_stride_g;
  u.st = st; u.term = st ? (double *)(ws + pl.off_term) : nullptr; u.term_stride = kTermStride; u.lloyd = lloyd; u.t = t;
  u.bimg = images ? (uint8_t *)(ws + pl.off_bimg) : nullptr;
  dim3 grid((unsigned)((K + kCPC - 1) / kCPC), (unsigned)v->G);
  DISPATCH_D(d, {
    GSRQ_CUDA_CHECK(cudaFuncSetAttribute(k_update<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)upd_smem_bytes<D>()));
    LAUNCH(kClsUpdate, stream, (k_update<D><<<grid, kUpdThreads, upd_smem_bytes<D>(), stream>>>(u)));
  });
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}


// ---- tensor-core scoring path (d == 16) ----
static bool use_tc(int d) {
  static const bool off = getenv("GSRQ_DISABLE_TC") != nullptr;
  return d == tc::kD && !off;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = []() -> EncodeTiledFn {
    void *f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
      return nullptr;
    return (EncodeTiledFn)f;
  }();
  return fn;
}

// 3-D tensor map over an operand plane [G][N][16] bf16: box = 128 rows of one group, SWIZZLE_32B,
// out-of-range rows read as zero.
static int make_plane_map(CUtensorMap *tm, const void *base, long long N, int G) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) { set_error("cuTensorMapEncodeTiled entry point not available"); return GSRQ_ECUDA; }
  const cuuint64_t dims[3] = {(cuuint64_t)tc::kD, (cuuint64_t)N, (cuuint64_t)G};
  const cuuint64_t strides[2] = {(cuuint64_t)tc::kD * 2, (cuuint64_t)N * tc::kD * 2};
  const cuuint32_t box[3] = {(cuuint32_t)tc::kD, (cuuint32_t)tc::kTileM, 1};
  const cuuint32_t es[3] = {1, 1, 1};
  CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(base), dims, strides, box, es,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed (%d)", (int)r); return GSRQ_ECUDA; }
  return GSRQ_OK;
}

struct TcMaps { CUtensorMap hi, lo; };

static int make_tc_maps(TcMaps *m, const Plan &pl, char *ws, int G, int n_planes) {
  int rc = make_plane_map(&m->hi, ws + pl.off_ahi, pl.Nf, G);
  if (rc) return rc;
  return make_plane_map(&m->lo, ws + (n_planes == 2 ? pl.off_alo : pl.off_ahi), pl.Nf, G);
}

// One assignment pass on the prepared fit rows: tcgen05 filter with the exact refine inside.
// The operand images (and max gain at gmax) of the scored codebook must already be in the workspace.
static int run_assign_tc(const Plan &pl, char *ws, const TcMaps &maps, int G, const float *shapes_st, const float *gains_st,
                         long long cb_stride_g, int K, int mode, int n_planes, uint8_t *idx, DevStats *st, int slot,
                         const int *gmax, long long gmax_stride, float *dbg, cudaStream_t stream) {
  tc::ScoreTcParams p{};
  p.bimg = (const uint8_t *)(ws + pl.off_bimg); p.gmax = gmax; p.gmax_stride = gmax_stride;
  p.rnorm = (const float *)(ws + pl.off_rnorm); p.rows = (const float *)(ws + pl.off_Rf);
  p.shapes = shapes_st; p.gains = gains_st; p.cb_stride_g = cb_stride_g; p.idx = idx; p.N = pl.Nf;
  p.n_tiles = (int)((pl.Nf + tc::kTileM - 1) / tc::kTileM); p.n_planes = n_planes; p.K = K; p.mode = mode;
  p.st = st; p.slot = slot; p.dbg = dbg;
  const int n_sm = sm_count();
  int ctas = n_sm / G; if (ctas < 1) ctas = 1; if (ctas > p.n_tiles) ctas = p.n_tiles;
  const size_t smem = 120 * 1024;  // > half of the SM's shared memory: one CTA (and one 512-column TMEM allocation) per SM
  static_assert(tc::kSmemTotal <= 120 * 1024, "smem budget");
  if (dbg) {
    GSRQ_CUDA_CHECK(cudaFuncSetAttribute(tc::k_score_tc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    LAUNCH(kClsScore, stream, (tc::k_score_tc<true><<<dim3((unsigned)ctas, (unsigned)G), tc::kThreads, smem, stream>>>(maps.hi, maps.lo, p)));
  } else {
    GSRQ_CUDA_CHECK(cudaFuncSetAttribute(tc::k_score_tc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    LAUNCH(kClsScore, stream, (tc::k_score_tc<false><<<dim3((unsigned)ctas, (unsigned)G), tc::kThreads, smem, stream>>>(maps.hi, maps.lo, p)));
  }
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

// The fused persistent fit kernel (k_fit_tc.cuh) on the prepared fit rows: passes [t_begin, t_end] of Alg. 1 in one
// cooperative launch, or (skip_scoring) one reduction + Eq. 7 / Eq. 8 update from the assignment already in `idx`.
static int run_fit_tc(const Plan &pl, char *ws, const TcMaps *maps, int G, int M, float *shapes_st, float *gains_st, long long cb_stride_g,
                      int K, int n_planes, uint8_t *idx, DevStats *st, int t_begin, int t_end, bool skip_scoring, int lloyd_override,
                      bool images, cudaStream_t stream) {
  tc::FitTcParams p{};
  p.bimg = images ? (uint8_t *)(ws + pl.off_bimg) : nullptr;
  p.shapes = shapes_st; p.gains = gains_st; p.cb_stride_g = cb_stride_g;
  p.rnorm = (const float *)(ws + pl.off_rnorm); p.rows = (const float *)(ws + pl.off_Rf);
  p.ahi = (const __nv_bfloat16 *)(ws + pl.off_ahi); p.wn = (const double *)(ws + pl.off_wn); p.wt = (const float *)(ws + pl.off_wt);
  p.nf_tok = pl.nf_tok; p.M = M; p.idx = idx; p.N = pl.Nf;
  p.n_tiles = (int)((pl.Nf + tc::kTileM - 1) / tc::kTileM); p.n_planes = n_planes; p.K = K;
  p.t_begin = t_begin; p.t_end = t_end; p.skip_scoring = skip_scoring ? 1 : 0; p.lloyd_override = lloyd_override;
  p.st = st; p.term = st ? (double *)(ws + pl.off_term) : nullptr; p.term_stride = kTermStride;
  p.part = (double *)(ws + pl.off_part); p.bar = (unsigned int *)(ws + pl.off_bar);
  p.chg = (uint2 *)(ws + pl.off_chg); p.chg_stride_g = pl.chg_stride_g;
  GSRQ_CUDA_CHECK(cudaMemsetAsync(p.bar, 0, (size_t)G * sizeof(unsigned int), stream));
  static const bool want_clk = getenv("GSRQ_FIT_CLOCKS") != nullptr;   // debug: per-phase cycle counts on stderr
  if (want_clk) {
    p.clk = (long long *)(ws + pl.off_clk);
    GSRQ_CUDA_CHECK(cudaMemsetAsync(p.clk, 0, (size_t)(G > kMaxCtas ? G : kMaxCtas) * 16 * sizeof(long long), stream));
  }
  const int n_sm = sm_count();
  int nx = n_sm / G; if (nx < 1) nx = 1; if (nx > p.n_tiles) nx = p.n_tiles;
  if ((long long)G * nx > kMaxCtas && nx > 1) nx = kMaxCtas / G > 0 ? kMaxCtas / G : 1;
  GSRQ_CUDA_CHECK(cudaFuncSetAttribute(tc::k_fit_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc::kFitSmemTotal));
  CUtensorMap zero;
  memset(&zero, 0, sizeof(zero));
  const CUtensorMap *hi = maps ? &maps->hi : &zero, *lo = maps ? &maps->lo : &zero;
  void *args[3] = {(void *)hi, (void *)lo, (void *)&p};
  const dim3 grid((unsigned)nx, (unsigned)G), block(tc::kThreads);
  {
    gsrq::ProfScope ps(skip_scoring ? kClsUpdate : kClsScore, stream);
    // nx > 1: the CTAs of a group wait on one another, so they must be co-resident: cooperative launch.  nx == 1: every
    // CTA is a group of its own (its barrier is trivially satisfied), any grid size is fine.
    if (nx > 1) GSRQ_CUDA_CHECK(cudaLaunchCooperativeKernel((const void *)tc::k_fit_tc, grid, block, args, tc::kFitSmemTotal, stream));
    else GSRQ_CUDA_CHECK(cudaLaunchKernel((const void *)tc::k_fit_tc, grid, block, args, tc::kFitSmemTotal, stream));
  }
  GSRQ_CUDA_CHECK(cudaGetLastError());
  if (want_clk) {
    std::vector<long long> h((size_t)G * nx * 16);
    GSRQ_CUDA_CHECK(cudaMemcpyAsync(h.data(), p.clk, h.size() * sizeof(long long), cudaMemcpyDeviceToHost, stream));
    GSRQ_CUDA_CHECK(cudaStreamSynchronize(stream));
    double sum[16] = {0};
    for (size_t c = 0; c < (size_t)G * nx; ++c) for (int q = 0; q < 16; ++q) sum[q] += (double)h[c * 16 + q];
    const double den = (double)G * nx * (t_end - t_begin + 1);
    fprintf(stderr, "k_fit_tc cycles per pass (mean over %d CTAs, %d passes): stage %.0f score %.0f reduce+publish %.0f bar1 %.0f merge %.0f bar2 %.0f | list entries %.0f batches %.1f; first-pass reduce %.0f cycles\n",
            G * nx, t_end - t_begin + 1, sum[0] / den, sum[1] / den, sum[2] / den, sum[3] / den, sum[4] / den, sum[5] / den, sum[6] / den, sum[7] / den,
            sum[8] / ((double)G * nx));
  }
  return GSRQ_OK;
}

static int launch_prep(const Plan &pl, const gsrq_view *v, const RowSrc &src, const float *w, long long w_stride_g,
                       const long long *fit_tokens, char *ws, bool consts, int n_planes, cudaStream_t stream) {
  PrepParams q{};
  q.src = src; q.w = w; q.w_stride_g = w_stride_g; q.fit_tokens = fit_tokens; q.nf_tok = pl.nf_tok;
  q.Rf = (float *)(ws + pl.off_Rf); q.wt = (float *)(ws + pl.off_wt);
  // the fused fit kernel (tensor-core path) reads w from wt and w/(||r||+eps) from wn; the cluster-owner update kernel reads pairs
  q.coef = use_tc(v->d) ? nullptr : (double2 *)(ws + pl.off_coef);
  q.wn = use_tc(v->d) ? (double *)(ws + pl.off_wn) : nullptr;
  q.epart = consts ? (double *)(ws + pl.off_epart) : nullptr;
  q.ahi = (consts && n_planes > 0) ? (__nv_bfloat16 *)(ws + pl.off_ahi) : nullptr;
  q.alo = (consts && n_planes == 2) ? (__nv_bfloat16 *)(ws + pl.off_alo) : nullptr;
  q.rnorm = (consts && n_planes > 0) ? (float *)(ws + pl.off_rnorm) : nullptr;
  dim3 grid((unsigned)pl.nE, (unsigned)v->G);
  const int d = v->d;
  LAUNCH(kClsPrep, stream, DISPATCH_D(d, (k_prep_rows<D><<<grid, 256, 0, stream>>>(q))));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

// Gather the fit rows (deriving the stage's residual when needed) with their per-row constants,
// operand planes (n_planes > 0) and energy partials.
static int prepare_rows(const Plan &pl, const void *kv, const gsrq_view *v, const float *w, long long w_stride_g,
                        const long long *fit_tokens, const gsrq_codebook *cb, int stage, const float *residual, char *ws,
                        cudaStream_t stream, int n_planes = 0) {
  const int d = v->d, G = v->G;
  float *Rf = (float *)(ws + pl.off_Rf);
  const bool derive = (!residual && stage > 0);
  int rc = launch_prep(pl, v, make_src(kv, v, residual, pl.Nall), w, w_stride_g, fit_tokens, ws, !derive, n_planes, stream);
  if (rc || !derive) return rc;
  // r = x - sum_{s<stage} c^(s)[a^(s)], in place on the compact rows; then the constants of the residual rows
  if (use_tc(d)) {  // tensor-core passes starting from the gathered fp32 rows (no codes wanted)
    rc = run_encode_tc(nullptr, v, Rf, pl.Nf, cb, stage, nullptr, 0, Rf, true, pl, ws, (unsigned int *)(ws + pl.off_cnt) + 200, stream);
    if (rc) return rc;
  } else {
    EncParams p{};
    p.src = make_src(nullptr, v, Rf, pl.Nf);
    p.N = pl.Nf; p.shapes = cb->shapes; p.gains = cb->gains; p.S = cb->S; p.K = cb->K;
    p.s_begin = 0; p.s_end = stage; p.s_base = 0; p.mode = 0; p.subtract = 1;
    p.codes = nullptr; p.code_stride_s = 0; p.res_out = Rf; p.st = nullptr; p.slot = 0;
    p.list = (uint2 *)(ws + pl.off_list);
    p.list_cnt = (unsigned int *)(ws + pl.off_cnt) + (kNumCounters - 1);
    rc = run_encode(p, G, d, stream);
    if (rc) return rc;
  }
  return launch_prep(pl, v, make_src(nullptr, v, Rf, pl.Nf), (const float *)(ws + pl.off_wt), pl.nf_tok, nullptr, ws, true,
                     n_planes, stream);
}

// ---- fused tensor-core encode (d == 16): passes of <= kEncMaxS stages ----
// The first pass reads a bf16 tensor straight through TMA; a dense fp32 tensor, and every later pass of a deep
// residual quantiser, start from fp32 rows (FROM_ROWS).
static bool can_encode_tc(const void *kv, const gsrq_view *v, int stage_begin) {
  const int M = v->hd / v->d;
  if (!use_tc(v->d) || stage_begin != 0 || ((uintptr_t)kv & 15) || v->T >= (1LL << 31)) return false;
  if (v->dtype == GSRQ_BF16) return M <= tc::kTileM && (M & (M - 1)) == 0;
  return v->stride_t == v->hd && v->stride_g == v->T * v->hd;  // fp32: the tensor itself is the [G][N][16] row buffer
}

// One pass: stages [s0, s0 + ns) of cb over N rows per group.  res_in == nullptr: rows come from the bf16 tensor kv.
static int run_encode_tc_pass(const void *kv, const gsrq_view *v, const gsrq_codebook *cb, int s0, int ns, long long N, uint8_t *codes,
                              long long code_stride_s, const float *res_in, float *res_out, const Plan &pl, char *ws,
                              unsigned int *list_cnt, cudaStream_t stream) {
  const int G = v->G, M = pl.M, tpt = tc::kTileM / (res_in ? 1 : M);
  CUtensorMap tm;
  memset(&tm, 0, sizeof(tm));
  bool head_inner = false;
  if (!res_in) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) { set_error("cuTensorMapEncodeTiled entry point not available"); return GSRQ_ECUDA; }
    // dims {16, M, T, G} (or {16, M, G, T} when the head stride is the smaller one); strides in bytes
    head_inner = v->stride_g < v->stride_t;
    const cuuint64_t dims[4] = {(cuuint64_t)tc::kD, (cuuint64_t)M, (cuuint64_t)(head_inner ? G : v->T), (cuuint64_t)(head_inner ? v->T : G)};
    const cuuint64_t strides[3] = {(cuuint64_t)tc::kD * 2, (cuuint64_t)(head_inner ? v->stride_g : v->stride_t) * 2,
                                   (cuuint64_t)(head_inner ? v->stride_t : v->stride_g) * 2};
    const cuuint32_t box[4] = {(cuuint32_t)tc::kD, (cuuint32_t)M, (cuuint32_t)(head_inner ? 1 : tpt), (cuuint32_t)(head_inner ? tpt : 1)};
    const cuuint32_t es[4] = {1, 1, 1, 1};
    CUresult r = fn(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void *>(kv), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled (kv) failed (%d)", (int)r); return GSRQ_ECUDA; }
  }
  uint8_t *bimg = (uint8_t *)(ws + pl.off_ebimg);
  int *gmax = (int *)(ws + pl.off_egmax);
  LAUNCH(kClsMisc, stream, (tc::k_bimg<<<G * ns, 256, 0, stream>>>(cb->shapes + (size_t)s0 * cb->K * tc::kD, cb->gains + (size_t)s0 * cb->K,
                                                                    (long long)cb->S * cb->K, ns, cb->K, 0, bimg, gmax)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  tc::EncTcParams p{};
  p.bimg = bimg; p.gmax = gmax; p.shapes = cb->shapes; p.gains = cb->gains; p.S = cb->S; p.K = cb->K; p.n_stages = ns; p.s0 = s0;
  p.res_in = res_in; p.codes = codes; p.code_stride_s = code_stride_s; p.res_out = res_out; p.N = N;
  p.n_tiles = (int)((N + tc::kTileM - 1) / tc::kTileM);
  if (!res_in) p.n_tiles = (int)((v->T + tpt - 1) / tpt);
  p.list = (uint2 *)(ws + pl.off_list); p.list_cnt = list_cnt;
  const int n_sm = sm_count();
  int ctas = n_sm / G; if (ctas < 1) ctas = 1; if (ctas > p.n_tiles) ctas = p.n_tiles;
  const size_t smem = tc::kEncSmemTotal;
  if (res_in) GSRQ_CUDA_CHECK(cudaFuncSetAttribute(tc::k_encode_tc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  else GSRQ_CUDA_CHECK(cudaFuncSetAttribute(tc::k_encode_tc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  if (res_in)
    LAUNCH(kClsEncode, stream, (tc::k_encode_tc<true><<<dim3((unsigned)ctas, (unsigned)G), tc::kThreads, smem, stream>>>(tm, p, tpt, 0)));
  else
    LAUNCH(kClsEncode, stream, (tc::k_encode_tc<false><<<dim3((unsigned)ctas, (unsigned)G), tc::kThreads, smem, stream>>>(tm, p, tpt, head_inner ? 1 : 0)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

// Stages [0, n_stages) over rows (kv through view, or the fp32 rows `rows0` [G][N][16] when kv == nullptr), in passes of
// kEncMaxS stages; after every pass the exact kernel finishes the rows the filter could not decide.  `carry` is the
// fp32 residual buffer between passes (and the result when the caller wants the residual); may alias rows0.
static int run_encode_tc(const void *kv, const gsrq_view *v, const float *rows0, long long N, const gsrq_codebook *cb, int n_stages,
                         uint8_t *codes, long long code_stride_s, float *carry, bool want_residual, const Plan &pl, char *ws,
                         unsigned int *cnt_base, cudaStream_t stream) {
  const int d = v->d;
  const float *cur = (kv && v->dtype == GSRQ_BF16) ? nullptr : (kv ? (const float *)kv : rows0);  // nullptr: TMA from the bf16 tensor
  int pass = 0;
  for (int s0 = 0; s0 < n_stages; s0 += tc::kEncMaxS, ++pass) {
    const int ns = (n_stages - s0 < tc::kEncMaxS) ? n_stages - s0 : tc::kEncMaxS;
    const bool last = s0 + ns == n_stages;
    float *out = (last && !want_residual) ? nullptr : carry;
    unsigned int *lc = cnt_base + pass;  // a fresh, zeroed counter per pass
    int rc = run_encode_tc_pass(kv, v, cb, s0, ns, N, codes, code_stride_s, cur, out, pl, ws, lc, stream);
    if (rc) return rc;
    EncParams e{};
    if (cur) e.src = make_src(nullptr, v, cur, N); else e.src = make_src(kv, v, nullptr, 0);
    e.N = N; e.shapes = cb->shapes; e.gains = cb->gains; e.S = cb->S; e.K = cb->K;
    e.s_first = s0; e.s_begin = s0; e.s_end = s0 + ns; e.s_base = 0; e.mode = 0; e.subtract = 1;
    e.codes = codes; e.code_stride_s = code_stride_s; e.res_out = out; e.st = nullptr; e.slot = 0;
    e.list = (uint2 *)(ws + pl.off_list); e.list_cnt = lc;
    LAUNCH(kClsRefine, stream, DISPATCH_D(d, (k_encode_exact<D><<<1184, 256, 0, stream>>>(e))));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    cur = carry;
  }
  return GSRQ_OK;
}


// ======================================================================================================================
// Wide sub-vectors (d = 64 / 128 / 256): exact fp64 kernels (k_wide.cuh) with the tcgen05 filter
// (k_score_tc_wide.cuh) in front of the assignment for d = 64 / 128.  One launch per step, stage by stage (unfused).
// ======================================================================================================================
struct WPlan {
  long long nf_tok, Nf, Nall, R, nE;   // R = rows the row-sized buffers hold
  int M;
  size_t off_st, off_cnt, off_rows, off_wt, off_wn, off_rnorm, off_idx, off_ids, off_epart, off_term, off_ahi, off_alo, off_bimg, off_gmax,
      off_list, off_part, off_starts, off_items, total;
};
constexpr int kWideParts = 4;   // row ranges per group in the wide update (k_wide.cuh)

// Sub-ranges of a group's rows for the stable counting sort in front of the wide update (k_wide_bucket): about 2048 rows each, at
// most 32 (larger ones for more rows); 0 = too many rows for that path, the update scans the assignment itself.
static int wide_nsub(long long N) {
  long long sub = 2048;
  while (sub < 32768 && (N + sub - 1) / sub > wide::kMaxSub) sub *= 2;
  const long long n = (N + sub - 1) / sub;
  if (n > wide::kMaxSub || N >= (1LL << 31)) return 0;
  return (int)n;
}
static long long wide_max_items(long long N, int K) { return N / wide::kItemRows + K + 1; }
static int wide_parts(long long N) { return (N >= 8192) ? kWideParts : 1; }

static bool wide_tc(int d) { return (d == 64 || d == 128) && use_tc(tc::kD); }

static WPlan make_wplan(const gsrq_view *v, long long n_fit_tokens) {
  WPlan p;
  p.M = v->hd / v->d;
  p.nf_tok = (n_fit_tokens > 0) ? n_fit_tokens : (n_fit_tokens == 0 ? v->T : 0);
  p.Nf = p.nf_tok * p.M;
  p.Nall = v->T * p.M;
  p.R = p.Nall;
  p.nE = (p.R + 7) / 8;
  const size_t G = (size_t)v->G, R = (size_t)p.R, d = (size_t)v->d;
  const bool tcp = wide_tc(v->d);
  size_t o = 0;
  p.off_st = o;    o += align_up(G * sizeof(DevStats));
  p.off_cnt = o;   o += align_up(kNumCounters * sizeof(unsigned int));
  p.off_rows = o;  o += align_up(G * R * d * sizeof(float));
  p.off_wt = o;    o += align_up(G * (size_t)v->T * sizeof(float));
  p.off_wn = o;    o += align_up(G * R * sizeof(double));
  p.off_rnorm = o; o += align_up(G * R * sizeof(float));
  p.off_idx = o;   o += align_up(G * R);
  p.off_ids = o;   o += align_up(G * GSRQ_MAX_K * sizeof(long long));
  p.off_epart = o; o += align_up(G * (size_t)p.nE * sizeof(double));
  p.off_term = o;  o += align_up(G * kTermStride * 256 * sizeof(double));
  p.off_ahi = o;   o += align_up(tcp ? G * R * d * 2 : 0);
  p.off_alo = o;   o += align_up(tcp ? G * R * d * 2 : 0);
  p.off_bimg = o;  o += align_up(tcp ? G * (size_t)tc::wide_bimg_bytes<2>() : 0);
  p.off_gmax = o;  o += align_up(G * sizeof(int));
  p.off_list = o;  o += align_up(G * R * sizeof(uint2));
  {
    const size_t scan_parts = (size_t)GSRQ_MAX_K * kWideParts, items = (size_t)wide_max_items(p.R, GSRQ_MAX_K);
    p.off_part = o;  o += align_up(G * (scan_parts > items ? scan_parts : items) * (2 * d + 2) * sizeof(double));
  }
  p.off_starts = o; o += align_up(G * (size_t)wide::kMaxSub * (GSRQ_MAX_K + 1) * sizeof(int));
  p.off_items = o;  o += align_up(G * (size_t)(GSRQ_MAX_K + 1) * sizeof(int));
  p.total = o;
  return p;
}

static int make_wide_map(CUtensorMap *tm, const void *base, long long N, int G, int d) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) { set_error("cuTensorMapEncodeTiled entry point not available"); return GSRQ_ECUDA; }
  const cuuint64_t dims[3] = {(cuuint64_t)d, (cuuint64_t)N, (cuuint64_t)G};
  const cuuint64_t strides[2] = {(cuuint64_t)d * 2, (cuuint64_t)N * d * 2};
  const cuuint32_t box[3] = {64, (cuuint32_t)tc::kTileM, 1};
  const cuuint32_t es[3] = {1, 1, 1};
  CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled (wide plane) failed (%d)", (int)r); return GSRQ_ECUDA; }
  return GSRQ_OK;
}

// gather (through fit_tokens) + per-row constants (+ operand planes) of N = nf_tok * M rows per group into the plan's row buffer
static int wide_prep(const WPlan &pl, const gsrq_view *v, const RowSrc &src, const float *w, long long w_stride_g, const long long *fit_tokens,
                     long long nf_tok, char *ws, bool planes, bool two_planes, bool energy, float *rows_out, cudaStream_t stream) {
  wide::WPrepParams q{};
  q.src = src; q.w = w; q.w_stride_g = w_stride_g; q.fit_tokens = fit_tokens; q.nf_tok = nf_tok;
  q.Rf = rows_out; q.wt = (float *)(ws + pl.off_wt); q.wn = (double *)(ws + pl.off_wn);
  q.rnorm = (float *)(ws + pl.off_rnorm);
  q.epart = energy ? (double *)(ws + pl.off_epart) : nullptr;
  q.ahi = planes ? (__nv_bfloat16 *)(ws + pl.off_ahi) : nullptr;
  q.alo = (planes && two_planes) ? (__nv_bfloat16 *)(ws + pl.off_alo) : nullptr;
  const long long N = nf_tok * src.M;
  dim3 grid((unsigned)((N + 7) / 8), (unsigned)v->G);
  LAUNCH(kClsPrep, stream, (wide::k_wide_prep<<<grid, 256, 0, stream>>>(q)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

// One assignment pass over N rows per group (rows fp32 [G][N][d]) against a stage slice: tcgen05 filter + exact kernel on the
// undecided rows (d = 64 / 128 with operand planes prepared), or the exact kernel on every row.
static int wide_assign(const WPlan &pl, const gsrq_view *v, char *ws, const float *rows, long long N, const float *shapes_st, const float *gains_st,
                       long long cb_stride_g, int K, int mode, bool use_filter, int n_planes, uint8_t *idx, DevStats *st, int slot,
                       unsigned int *list_cnt, float *dbg, cudaStream_t stream) {
  const int G = v->G, d = v->d;
  wide::WAssignParams a{};
  a.rows = rows; a.N = N; a.d = d; a.K = K; a.mode = mode; a.shapes = shapes_st; a.gains = gains_st; a.cb_stride_g = cb_stride_g;
  a.idx = idx; a.idx16 = 0; a.st = st; a.slot = slot;
  const size_t smem = wide::wide_assign_smem(d);
  GSRQ_CUDA_CHECK(cudaFuncSetAttribute(wide::k_wide_assign, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  if (!use_filter) {
    dim3 grid((unsigned)((N + wide::kWaRows - 1) / wide::kWaRows), (unsigned)G);
    LAUNCH(kClsRefine, stream, (wide::k_wide_assign<<<grid, 256, smem, stream>>>(a)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    return GSRQ_OK;
  }
  uint8_t *bimg = (uint8_t *)(ws + pl.off_bimg);
  int *gmax = (int *)(ws + pl.off_gmax);
  uint2 *list = (uint2 *)(ws + pl.off_list);
  GSRQ_CUDA_CHECK(cudaMemsetAsync(list_cnt, 0, sizeof(unsigned int), stream));
  GSRQ_CUDA_CHECK(cudaMemsetAsync(gmax, 0, (size_t)G * sizeof(int), stream));
  CUtensorMap tmh, tml;
  int rc = make_wide_map(&tmh, ws + pl.off_ahi, N, G, d);
  if (rc) return rc;
  rc = make_wide_map(&tml, ws + (n_planes == 2 ? pl.off_alo : pl.off_ahi), N, G, d);
  if (rc) return rc;
  tc::ScoreWideParams p{};
  p.bimg = bimg; p.gmax = gmax; p.rnorm = (const float *)(ws + pl.off_rnorm); p.gains = gains_st; p.cb_stride_g = cb_stride_g;
  p.idx = idx; p.N = N; p.n_tiles = (int)((N + tc::kTileM - 1) / tc::kTileM); p.n_planes = n_planes; p.K = K; p.mode = (mode == wide::kModeProj) ? 1 : 0;
  p.st = st; p.slot = slot; p.list = list; p.list_cnt = list_cnt; p.dbg = dbg;
  const int n_sm = sm_count();
  int ctas = n_sm / G; if (ctas < 1) ctas = 1; if (ctas > p.n_tiles) ctas = p.n_tiles;
  const dim3 grid((unsigned)ctas, (unsigned)G);
#define GSRQ_WIDE_TC(KB, DBG)                                                                                                                   \
  do {                                                                                                                                          \
    LAUNCH(kClsMisc, stream, (tc::k_bimg_wide<KB><<<dim3((unsigned)G, 8), 256, 0, stream>>>(shapes_st, gains_st, cb_stride_g, K, p.mode, bimg, gmax))); \
    GSRQ_CUDA_CHECK(cudaGetLastError());                                                                                                        \
    GSRQ_CUDA_CHECK(cudaFuncSetAttribute(tc::k_score_tc_wide<KB, DBG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc::WideSmem<KB>::kTotal)); \
    LAUNCH(kClsScore, stream, (tc::k_score_tc_wide<KB, DBG><<<grid, tc::kThreads, tc::WideSmem<KB>::kTotal, stream>>>(tmh, tml, p)));             \
  } while (0)
  if (d == 128) { if (dbg) GSRQ_WIDE_TC(2, true); else GSRQ_WIDE_TC(2, false); }
  else { if (dbg) GSRQ_WIDE_TC(1, true); else GSRQ_WIDE_TC(1, false); }
#undef GSRQ_WIDE_TC
  GSRQ_CUDA_CHECK(cudaGetLastError());
  a.list_cnt = list_cnt;
  // the list length is only known on the device: a machine-filling grid strides over it (one warp per undecided row)
  LAUNCH(kClsRefine, stream, (wide::k_wide_refine<<<2 * n_sm, 256, (size_t)8 * d * sizeof(double), stream>>>(a, list)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

static int wide_subtract(const WPlan &pl, const gsrq_view *v, char *ws, float *rows, long long N, const float *shapes_st, const float *gains_st,
                         long long cb_stride_g, int K, const uint8_t *idx, uint8_t *codes, bool planes, cudaStream_t stream) {
  wide::WSubParams q{};
  q.rows = rows; q.N = N; q.d = v->d; q.K = K; q.shapes = shapes_st; q.gains = gains_st; q.cb_stride_g = cb_stride_g; q.idx = idx; q.codes = codes;
  q.ahi = planes ? (__nv_bfloat16 *)(ws + pl.off_ahi) : nullptr; q.alo = planes ? (__nv_bfloat16 *)(ws + pl.off_alo) : nullptr;
  q.rnorm = planes ? (float *)(ws + pl.off_rnorm) : nullptr;
  dim3 grid((unsigned)((N + 7) / 8), (unsigned)v->G);
  LAUNCH(kClsEncode, stream, (wide::k_wide_subtract<<<grid, 256, 0, stream>>>(q)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

static int wide_update(const WPlan &pl, const gsrq_view *v, char *ws, const float *rows, long long N, long long nf_tok, const uint8_t *idx,
                       float *shapes_st, float *gains_st, long long cb_stride_g, int K, int mode, DevStats *st, int t, cudaStream_t stream) {
  wide::WUpdateParams u{};
  u.rows = rows; u.wn = (const double *)(ws + pl.off_wn); u.wt = (const float *)(ws + pl.off_wt); u.nf_tok = nf_tok; u.M = pl.M;
  u.idx = idx; u.idx16 = 0; u.N = N; u.d = v->d; u.K = K; u.shapes = shapes_st; u.gains = gains_st; u.cb_stride_g = cb_stride_g; u.mode = mode;
  u.st = st; u.term = st ? (double *)(ws + pl.off_term) : nullptr; u.term_stride = kTermStride; u.term_k = 256; u.t = t; u.gmax = nullptr;
  u.part = (double *)(ws + pl.off_part);
  u.nsub = wide_nsub(N);
  if (u.nsub > 0) {
    // rows sorted by cluster (the undecided-row list of the assignment is free by now and holds the order), then balanced items
    wide::WBucketParams b{};
    b.idx = idx; b.N = N; b.K = K; b.nsub = u.nsub; b.order = (int *)(ws + pl.off_list); b.starts = (int *)(ws + pl.off_starts); b.st = st; b.t = t;
    const size_t bsmem = (size_t)256 * K * sizeof(uint16_t);
    GSRQ_CUDA_CHECK(cudaFuncSetAttribute(wide::k_wide_bucket, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bsmem));
    LAUNCH(kClsUpdate, stream, (wide::k_wide_bucket<<<dim3((unsigned)u.nsub, (unsigned)v->G), 256, bsmem, stream>>>(b)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    u.order = b.order; u.starts = b.starts; u.item_first = (int *)(ws + pl.off_items); u.max_items = (int)wide_max_items(N, K); u.nparts = 1;
    LAUNCH(kClsUpdate, stream, (wide::k_wide_items<<<(unsigned)v->G, 256, 0, stream>>>(u)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    const dim3 igrid((unsigned)((u.max_items + 7) / 8), (unsigned)v->G);
    if (v->d > 128) LAUNCH(kClsUpdate, stream, (wide::k_wide_update_items<2><<<igrid, 256, 0, stream>>>(u)));
    else LAUNCH(kClsUpdate, stream, (wide::k_wide_update_items<1><<<igrid, 256, 0, stream>>>(u)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    LAUNCH(kClsUpdate, stream, (wide::k_wide_update_items_finish<<<dim3((unsigned)K, (unsigned)v->G), 256, 0, stream>>>(u)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    return GSRQ_OK;
  }
  u.nparts = wide_parts(N);
  const dim3 ugrid((unsigned)K, (unsigned)v->G, (unsigned)u.nparts);
  const size_t usmem = wide::wide_update_smem();
  if (v->d > 128) LAUNCH(kClsUpdate, stream, (wide::k_wide_update<2><<<ugrid, 256, usmem, stream>>>(u)));
  else LAUNCH(kClsUpdate, stream, (wide::k_wide_update<1><<<ugrid, 256, usmem, stream>>>(u)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  if (u.nparts > 1) {
    LAUNCH(kClsUpdate, stream, (wide::k_wide_update_finish<<<dim3((unsigned)K, (unsigned)v->G), 256, 0, stream>>>(u)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
  }
  return GSRQ_OK;
}

// rows of the fit (gathered through fit_tokens; the stage's residual derived from kv + earlier stages when not given)
static int wide_fit_rows(const WPlan &pl, const void *kv, const gsrq_view *v, const float *w, long long w_stride_g, const long long *fit_tokens,
                         const gsrq_codebook *cb, int stage, const float *residual, char *ws, bool planes, int n_planes, cudaStream_t stream) {
  float *Rf = (float *)(ws + pl.off_rows);
  const bool derive = (!residual && stage > 0);
  const int K = cb ? cb->K : 0, d = v->d;
  int rc = wide_prep(pl, v, make_src(kv, v, residual, pl.Nall), w, w_stride_g, fit_tokens, pl.nf_tok, ws, planes && !derive, n_planes == 2, !derive, Rf, stream);
  if (rc || !derive) return rc;
  uint8_t *idx = (uint8_t *)(ws + pl.off_idx);
  unsigned int *cnt = (unsigned int *)(ws + pl.off_cnt);
  for (int s = 0; s < stage; ++s) {   // r = x - sum_{s < stage} c^(s)[a^(s)] on the compact rows, stage by stage (exact kernel: no planes yet)
    const float *sh = cb->shapes + (size_t)s * K * d, *ga = cb->gains + (size_t)s * K;
    rc = wide_assign(pl, v, ws, Rf, pl.Nf, sh, ga, (long long)cb->S * K, K, wide::kModeGskm, false, 2, idx, nullptr, 0, cnt + 200 + s, nullptr, stream);
    if (rc) return rc;
    rc = wide_subtract(pl, v, ws, Rf, pl.Nf, sh, ga, (long long)cb->S * K, K, idx, nullptr, false, stream);
    if (rc) return rc;
  }
  GSRQ_CUDA_CHECK(cudaMemsetAsync(idx, 0, (size_t)v->G * pl.Nf, stream));
  // per-row constants of the residual rows; weights come from the compact per-fit-token array written by the first pass
  wide::WPrepParams q{};
  q.src = make_src(nullptr, v, Rf, pl.Nf); q.w = (const float *)(ws + pl.off_wt); q.w_stride_g = pl.nf_tok; q.fit_tokens = nullptr; q.nf_tok = pl.nf_tok;
  q.Rf = Rf; q.wt = (float *)(ws + pl.off_wt); q.wn = (double *)(ws + pl.off_wn); q.rnorm = (float *)(ws + pl.off_rnorm);
  q.epart = (double *)(ws + pl.off_epart);
  q.ahi = planes ? (__nv_bfloat16 *)(ws + pl.off_ahi) : nullptr; q.alo = (planes && n_planes == 2) ? (__nv_bfloat16 *)(ws + pl.off_alo) : nullptr;
  dim3 grid((unsigned)((pl.Nf + 7) / 8), (unsigned)v->G);
  LAUNCH(kClsPrep, stream, (wide::k_wide_prep<<<grid, 256, 0, stream>>>(q)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

static int fit_stage_wide(const void *kv, const gsrq_view *view, const float *w, int64_t w_stride_g, const int64_t *fit_tokens, int64_t n_fit,
                          gsrq_codebook *cb, int stage, const float *residual, int iters, uint64_t seed, gsrq_fit_stats *stats, void *workspace,
                          size_t workspace_bytes, cudaStream_t stream) {
  const WPlan pl = make_wplan(view, fit_tokens ? n_fit : 0);
  if (pl.Nf < cb->K) { set_error("fewer fit rows (%lld) than codewords (%d)", pl.Nf, cb->K); return GSRQ_EDEGENERATE; }
  int rc = check_ws(workspace, workspace_bytes, pl.total);
  if (rc) return rc;
  char *ws = (char *)workspace;
  const int G = view->G, d = view->d, K = cb->K;
  DevStats *st = (DevStats *)(ws + pl.off_st);
  unsigned int *cnt = (unsigned int *)(ws + pl.off_cnt);
  uint8_t *idx = (uint8_t *)(ws + pl.off_idx);
  float *Rf = (float *)(ws + pl.off_rows);
  GSRQ_CUDA_CHECK(cudaMemsetAsync(st, 0, (size_t)G * sizeof(DevStats), stream));
  GSRQ_CUDA_CHECK(cudaMemsetAsync(cnt, 0, kNumCounters * sizeof(unsigned int), stream));
  GSRQ_CUDA_CHECK(cudaMemsetAsync(idx, 0, (size_t)G * pl.Nf, stream));
  const bool filter = wide_tc(d);
  const int n_planes = (stage == 0 && !residual && view->dtype == GSRQ_BF16) ? 1 : 2;
  rc = wide_fit_rows(pl, kv, view, w, w_stride_g, (const long long *)fit_tokens, cb, stage, residual, ws, filter, n_planes, stream);
  if (rc) return rc;
  float *shapes_st = cb->shapes + (size_t)stage * K * d;
  float *gains_st = cb->gains + (size_t)stage * K;
  const long long cb_stride_g = (long long)cb->S * K;
  LAUNCH(kClsPrep, stream, (wide::k_wide_init<<<G, 512, (size_t)K * sizeof(long long), stream>>>(Rf, pl.Nf, d, K, G, stage, seed, (long long *)(ws + pl.off_ids), st,
                                                                                                shapes_st, gains_st, cb_stride_g, 0)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  for (int t = 0; t <= iters; ++t) {   // t = 0: Alg. 1 l.2 (gains under the max-projection assignment); t >= 1: Lloyd iterations
    rc = wide_assign(pl, view, ws, Rf, pl.Nf, shapes_st, gains_st, cb_stride_g, K, t == 0 ? wide::kModeProj : wide::kModeGskm, filter, n_planes, idx, st, t,
                     cnt + (t % 128), nullptr, stream);
    if (rc) return rc;
    rc = wide_update(pl, view, ws, Rf, pl.Nf, pl.nf_tok, idx, shapes_st, gains_st, cb_stride_g, K, t > 0 ? 1 : 0, st, t, stream);
    if (rc) return rc;
    LAUNCH(kClsMisc, stream, (wide::k_wide_converged<<<(G + 255) / 256, 256, 0, stream>>>(st, G, t)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
  }
  if (!stats) return GSRQ_OK;
  LAUNCH(kClsMisc, stream, (k_finish<<<G, 160, 0, stream>>>(st, (const double *)(ws + pl.off_term), kTermStride, K, (const double *)(ws + pl.off_epart),
                                                            (int)((pl.Nf + 7) / 8), iters)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;   // the caller copies the statistics
}

static int encode_wide(const void *kv, const gsrq_view *view, const gsrq_codebook *cb, int stage_begin, int stage_end, uint8_t *codes,
                       float *residual_out, void *workspace, size_t workspace_bytes, cudaStream_t stream) {
  const WPlan pl = make_wplan(view, -1);
  int rc = check_ws(workspace, workspace_bytes, pl.total);
  if (rc) return rc;
  char *ws = (char *)workspace;
  const int G = view->G, d = view->d, K = cb->K;
  const long long N = pl.Nall, cb_stride_g = (long long)cb->S * K;
  unsigned int *cnt = (unsigned int *)(ws + pl.off_cnt);
  float *R = residual_out ? residual_out : (float *)(ws + pl.off_rows);
  const bool filter = wide_tc(d);
  // the working residual: all rows of kv as fp32 (+ the bf16-exact operand plane when stage 0 is scored by the filter)
  rc = wide_prep(pl, view, make_src(kv, view, nullptr, 0), nullptr, 0, nullptr, view->T, ws, filter && stage_begin == 0, view->dtype != GSRQ_BF16, false, R, stream);
  if (rc) return rc;
  for (int s = 0; s < stage_end; ++s) {
    const float *sh = cb->shapes + (size_t)s * K * d, *ga = cb->gains + (size_t)s * K;
    uint8_t *plane = codes + (size_t)s * G * N;
    if (s >= stage_begin) {
      const int n_planes = (s == 0 && view->dtype == GSRQ_BF16) ? 1 : 2;
      rc = wide_assign(pl, view, ws, R, N, sh, ga, cb_stride_g, K, wide::kModeGskm, filter, n_planes, plane, nullptr, 0, cnt + 1 + (s % 64), nullptr, stream);
      if (rc) return rc;
    }
    const bool need_res = (s + 1 < stage_end) || residual_out;
    if (!need_res) break;
    // planes of the new residual only when the next stage is scored by the filter
    rc = wide_subtract(pl, view, ws, R, N, sh, ga, cb_stride_g, K, plane, nullptr, filter && s + 1 < stage_end && s + 1 >= stage_begin, stream);
    if (rc) return rc;
  }
  return GSRQ_OK;
}

static int decode_wide(const uint8_t *codes, const gsrq_codebook *cb, int n_stages, void *kv_out, const gsrq_view *ov, cudaStream_t stream) {
  wide::WDecParams p{};
  p.codes = codes; p.shapes = cb->shapes; p.gains = cb->gains; p.S = cb->S; p.K = cb->K; p.G = ov->G; p.n_stages = n_stages; p.d = ov->d;
  p.M = ov->hd / ov->d; p.N = ov->T * p.M; p.out = kv_out; p.dtype = ov->dtype; p.stride_g = ov->stride_g; p.stride_t = ov->stride_t;
  dim3 grid((unsigned)((p.N + 7) / 8), (unsigned)ov->G);
  LAUNCH(kClsDecode, stream, (wide::k_wide_decode<<<grid, 256, 0, stream>>>(p)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

// ---- stand-alone clustering of fp32 rows: GSKM (Alg. 1) or textbook weighted K-means, one group, K <= 4096 ----
struct CPlan { size_t off_st, off_rows, off_wt, off_wn, off_rnorm, off_idx, off_ids, off_epart, off_term, off_part, off_met, total; long long nE; };

static CPlan make_cplan(long long N, int d, int K) {
  CPlan p;
  size_t o = 0;
  p.nE = (N + 7) / 8;
  p.off_st = o;    o += align_up(sizeof(DevStats));
  p.off_rows = o;  o += align_up((size_t)N * d * sizeof(float));
  p.off_wt = o;    o += align_up((size_t)N * sizeof(float));
  p.off_wn = o;    o += align_up((size_t)N * sizeof(double));
  p.off_rnorm = o; o += align_up((size_t)N * sizeof(float));
  p.off_idx = o;   o += align_up((size_t)N * sizeof(uint16_t));
  p.off_ids = o;   o += align_up((size_t)K * sizeof(long long));
  p.off_epart = o; o += align_up((size_t)p.nE * sizeof(double));
  p.off_term = o;  o += align_up((size_t)kTermStride * K * sizeof(double));
  p.off_part = o;  o += align_up((size_t)K * kWideParts * (2 * d + 2) * sizeof(double));
  p.off_met = o;   o += align_up((size_t)p.nE * 5 * sizeof(double) + 64);
  p.total = o;
  return p;
}

static int check_cluster(long long N, int d, int K) {
  if (N <= 0 || d <= 0 || d > wide::kMaxD || (d & 3) || K <= 0 || K > wide::kMaxK) {
    set_error("clustering: need N > 0, d a multiple of 4 in [4, %d], K in [1, %d] (got N=%lld d=%d K=%d)", wide::kMaxD, wide::kMaxK, N, d, K);
    return GSRQ_EINVAL;
  }
  return GSRQ_OK;
}

static int cluster_assign(const float *rows, long long N, int d, int K, int mode, const float *shapes, const float *gains, uint16_t *idx, DevStats *st,
                          int slot, cudaStream_t stream) {
  wide::WAssignParams a{};
  a.rows = rows; a.N = N; a.d = d; a.K = K; a.mode = mode; a.shapes = shapes; a.gains = gains; a.cb_stride_g = K; a.idx = idx; a.idx16 = 1;
  a.st = st; a.slot = slot;
  const size_t smem = wide::wide_assign_smem(d);
  GSRQ_CUDA_CHECK(cudaFuncSetAttribute(wide::k_wide_assign, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  LAUNCH(kClsRefine, stream, (wide::k_wide_assign<<<dim3((unsigned)((N + wide::kWaRows - 1) / wide::kWaRows), 1), 256, smem, stream>>>(a)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

}  // namespace gsrq

using namespace gsrq;

// Copy the device statistics of a fit to the caller's host structs (synchronises the stream).
static int copy_fit_stats(const DevStats *st, int G, gsrq_fit_stats *stats, cudaStream_t stream) {
  {
    DevStats *h = (DevStats *)malloc((size_t)G * sizeof(DevStats));
    if (!h) { set_error("out of host memory"); return GSRQ_ECUDA; }
    cudaError_t e = cudaMemcpyAsync(h, st, (size_t)G * sizeof(DevStats), cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) { free(h); set_error("stats copy failed: %s", cudaGetErrorString(e)); return GSRQ_ECUDA; }
    int degenerate = 0, lost = 0;
    for (int g = 0; g < G; ++g) {
      gsrq_fit_stats *o = stats + g;
      memset(o, 0, sizeof(*o));
      o->iters_run = h[g].iters_run;
      o->n_refined = h[g].refined;
      for (int t = 1; t <= h[g].iters_run; ++t) {
        o->wdist_after_assign[t - 1] = h[g].J[t];
        o->n_changed[t - 1] = h[g].changed[t];
      }
      o->n_empty_last = h[g].n_empty[h[g].iters_run];
      o->n_changed_last = h[g].iters_run ? h[g].changed[h[g].iters_run] : 0;
      degenerate |= (h[g].err == GSRQ_EDEGENERATE);
      lost |= (h[g].err != 0 && h[g].err != GSRQ_EDEGENERATE);
    }
    free(h);
    if (lost) { set_error("the fit kernel's group barrier timed out"); return GSRQ_ECUDA; }
    if (degenerate) { set_error("a group has fewer than K distinct non-zero fit rows"); return GSRQ_EDEGENERATE; }
  }
  return GSRQ_OK;
}

extern "C" {

const char *gsrq_last_error(void) { return g_err; }
const char *gsrq_version(void) { return "gsrq-b200 0.1 (sm_100a)"; }

size_t gsrq_workspace_bytes(const gsrq_view *view, int K, int S, int64_t n_fit_tokens) {
  if (check_view(view, K, S) != GSRQ_OK) return 0;
  if (n_fit_tokens > view->T) { set_error("n_fit_tokens > T"); return 0; }
  if (is_wide(view->d)) return make_wplan(view, n_fit_tokens).total;
  return make_plan(view, K, S, n_fit_tokens).total;
}

int gsrq_fit_stage(const void *kv, const gsrq_view *view, const float *w, int64_t w_stride_g, const int64_t *fit_tokens,
                   int64_t n_fit, gsrq_codebook *cb, int stage, const float *residual, int iters, uint64_t seed,
                   gsrq_fit_stats *stats, void *workspace, size_t workspace_bytes, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!kv || !cb || !cb->shapes || !cb->gains) { set_error("NULL kv / codebook"); return GSRQ_EINVAL; }
  int rc = check_view(view, cb->K, cb->S);
  if (rc) return rc;
  if (stage < 0 || stage >= cb->S) { set_error("stage %d out of [0, %d)", stage, cb->S); return GSRQ_EINVAL; }
  if (iters < 0 || iters > GSRQ_MAX_ITERS) { set_error("iters must be in [0, %d]", GSRQ_MAX_ITERS); return GSRQ_EINVAL; }
  if (fit_tokens && (n_fit <= 0 || n_fit > view->T)) { set_error("n_fit out of range"); return GSRQ_EINVAL; }
  if ((rc = check_align16(kv, "kv")) || (rc = check_align16(residual, "residual"))) return rc;
  if (is_wide(view->d)) {
    rc = fit_stage_wide(kv, view, w, w_stride_g, fit_tokens, n_fit, cb, stage, residual, iters, seed, stats, workspace, workspace_bytes, stream);
    if (rc || !stats) return rc;
    return copy_fit_stats((const DevStats *)((char *)workspace + make_wplan(view, fit_tokens ? n_fit : 0).off_st), view->G, stats, stream);
  }
  const Plan pl = make_plan(view, cb->K, cb->S, fit_tokens ? n_fit : 0);
  if (pl.Nf < cb->K) { set_error("fewer fit rows (%lld) than codewords (%d)", pl.Nf, cb->K); return GSRQ_EDEGENERATE; }
  rc = check_ws(workspace, workspace_bytes, pl.total);
  if (rc) return rc;
  char *ws = (char *)workspace;
  const int G = view->G, d = view->d, K = cb->K;
  DevStats *st = (DevStats *)(ws + pl.off_st);
  unsigned int *cnt = (unsigned int *)(ws + pl.off_cnt);
  uint8_t *idx = (uint8_t *)(ws + pl.off_idx);
  long long *ids = (long long *)(ws + pl.off_ids);
  float *Rf = (float *)(ws + pl.off_Rf);
  GSRQ_CUDA_CHECK(cudaMemsetAsync(st, 0, (size_t)G * sizeof(DevStats), stream));
  GSRQ_CUDA_CHECK(cudaMemsetAsync(cnt, 0, kNumCounters * sizeof(unsigned int), stream));
  GSRQ_CUDA_CHECK(cudaMemsetAsync(idx, 0, (size_t)G * pl.Nf, stream));
  // rows are bf16-exact only for stage 0 of a bf16 tensor; otherwise the A operand is split hi + lo
  const int n_planes = !use_tc(d) ? 0 : ((stage == 0 && !residual && view->dtype == GSRQ_BF16) ? 1 : 2);
  rc = prepare_rows(pl, kv, view, w, w_stride_g, (const long long *)fit_tokens, cb, stage, residual, ws, stream, n_planes);
  if (rc) return rc;

  float *shapes_st = cb->shapes + (size_t)stage * K * d;
  float *gains_st = cb->gains + (size_t)stage * K;
  const long long cb_stride_g = (long long)cb->S * K;
  uint8_t *bimg = n_planes ? (uint8_t *)(ws + pl.off_bimg) : nullptr;
  LAUNCH(kClsPrep, stream, DISPATCH_D(d, (k_init_ids<D><<<G, 512, 0, stream>>>(Rf, pl.Nf, K, G, stage, seed, ids, st, shapes_st, gains_st,
                                                                              cb_stride_g, bimg))));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  TcMaps maps;
  if (n_planes) { rc = make_tc_maps(&maps, pl, ws, G, n_planes); if (rc) return rc; }

  EncParams p{};
  p.src = make_src(nullptr, view, Rf, pl.Nf);
  p.N = pl.Nf; p.S = cb->S; p.K = K;
  p.subtract = 0;
  p.codes = idx; p.code_stride_s = 0; p.res_out = nullptr; p.st = st;
  p.list = (uint2 *)(ws + pl.off_list);
  // score only stage `stage` on the prepared rows: present it to the kernels as a 1-stage pass
  p.shapes = shapes_st; p.gains = gains_st; p.s_begin = 0; p.s_end = 1; p.s_base = 0;
  // t = 0 is Alg. 1 l.2: gains by Eq. 8 under the max-projection assignment (reading c-I);
  // t >= 1 are the Lloyd iterations.  Two launches per pass: assignment, then the fused update.
  if (n_planes) {  // d == 16: the whole loop is one persistent kernel (k_fit_tc.cuh)
    rc = run_fit_tc(pl, ws, &maps, G, pl.M, shapes_st, gains_st, cb_stride_g, K, n_planes, idx, st, 0, iters, false, -1, true, stream);
  } else {
    for (int t = 0; t <= iters && rc == 0; ++t) {
      EncParams a = p;
      a.mode = (t == 0) ? 1 : 0; a.slot = t; a.list_cnt = cnt + t;
      rc = run_encode(a, G, d, stream);
      if (rc) break;
      rc = run_update(pl, view, K, ws, idx, shapes_st, gains_st, cb_stride_g, st, t > 0, t, false, stream);
    }
  }
  if (rc) return rc;
  if (stats) {  // J_t and iters_run are only read back through `stats`
    LAUNCH(kClsMisc, stream, (k_finish<<<G, 160, 0, stream>>>(st, (const double *)(ws + pl.off_term), kTermStride, K,
                                                              (const double *)(ws + pl.off_epart), (int)pl.nE, iters)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
  }
  if (stats) return copy_fit_stats(st, G, stats, stream);
  return GSRQ_OK;
}

int gsrq_fit_status(const void *workspace, const gsrq_view *view, int K, int S, int64_t n_fit_tokens, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!workspace) { set_error("workspace is NULL"); return GSRQ_EINVAL; }
  int rc = check_view(view, K, S);
  if (rc) return rc;
  if (n_fit_tokens < 0 || n_fit_tokens > view->T) { set_error("n_fit_tokens out of [0, T]"); return GSRQ_EINVAL; }
  const size_t off = is_wide(view->d) ? make_wplan(view, n_fit_tokens).off_st : make_plan(view, K, S, n_fit_tokens).off_st;
  const DevStats *st = (const DevStats *)((const char *)workspace + off);
  std::vector<int> err((size_t)view->G, 0);
  // the G error words, one per DevStats record
  GSRQ_CUDA_CHECK(cudaMemcpy2DAsync(err.data(), sizeof(int), &st[0].err, sizeof(DevStats), sizeof(int), (size_t)view->G, cudaMemcpyDeviceToHost, stream));
  GSRQ_CUDA_CHECK(cudaStreamSynchronize(stream));
  bool degenerate = false;
  for (int g = 0; g < view->G; ++g) {
    if (err[g] == GSRQ_EDEGENERATE) degenerate = true;
    else if (err[g] != 0) { set_error("the fit kernel's group barrier timed out (group %d): the codebook of this stage is not valid", g); return GSRQ_ECUDA; }
  }
  if (degenerate) { set_error("a group has fewer than K distinct non-zero fit rows"); return GSRQ_EDEGENERATE; }
  return GSRQ_OK;
}


int gsrq_encode(const void *kv, const gsrq_view *view, const gsrq_codebook *cb, int stage_begin, int stage_end,
                uint8_t *codes, float *residual_out, void *workspace, size_t workspace_bytes, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!kv || !cb || !cb->shapes || !cb->gains || !codes) { set_error("NULL kv / codebook / codes"); return GSRQ_EINVAL; }
  int rc = check_view(view, cb->K, cb->S);
  if (rc) return rc;
  if (stage_begin < 0 || stage_end > cb->S || stage_begin >= stage_end) { set_error("bad stage range [%d, %d)", stage_begin, stage_end); return GSRQ_EINVAL; }
  if ((rc = check_align16(kv, "kv")) || (rc = check_align16(residual_out, "residual_out"))) return rc;
  if (is_wide(view->d)) return encode_wide(kv, view, cb, stage_begin, stage_end, codes, residual_out, workspace, workspace_bytes, stream);
  const Plan pl = make_plan(view, cb->K, cb->S, -1);
  rc = check_ws(workspace, workspace_bytes, pl.encode_total);
  if (rc) return rc;
  char *ws = (char *)workspace;
  unsigned int *cnt = (unsigned int *)(ws + pl.off_cnt);
  GSRQ_CUDA_CHECK(cudaMemsetAsync(cnt, 0, 16 * sizeof(unsigned int), stream));
  EncParams p{};
  p.src = make_src(kv, view, nullptr, 0);
  p.N = pl.Nall; p.shapes = cb->shapes; p.gains = cb->gains; p.S = cb->S; p.K = cb->K;
  p.s_begin = stage_begin; p.s_end = stage_end; p.s_base = 0; p.mode = 0; p.subtract = 1;
  p.codes = codes; p.code_stride_s = (long long)view->G * pl.Nall; p.res_out = residual_out;
  p.st = nullptr; p.slot = 0; p.list = (uint2 *)(ws + pl.off_list); p.list_cnt = cnt;
  if (can_encode_tc(kv, view, stage_begin)) {
    // tensor-core passes of <= 4 stages; after each, the exact kernel finishes the rows the filter could not decide
    float *carry = residual_out ? residual_out : (float *)(ws + pl.off_eres);
    return run_encode_tc(kv, view, nullptr, pl.Nall, cb, stage_end, codes, (long long)view->G * pl.Nall, carry, residual_out != nullptr, pl, ws,
                         cnt, stream);
  }
  return run_encode(p, view->G, view->d, stream);
}

int gsrq_decode(const uint8_t *codes, const gsrq_codebook *cb, int n_stages, void *kv_out, const gsrq_view *out_view,
                gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!codes || !cb || !cb->shapes || !cb->gains || !kv_out) { set_error("NULL codes / codebook / output"); return GSRQ_EINVAL; }
  int rc = check_view(out_view, cb->K, cb->S);
  if (rc) return rc;
  if (n_stages < 0 || n_stages > cb->S) { set_error("n_stages %d out of [0, %d]", n_stages, cb->S); return GSRQ_EINVAL; }
  if ((rc = check_align16(kv_out, "kv_out"))) return rc;
  if (is_wide(out_view->d)) return decode_wide(codes, cb, n_stages, kv_out, out_view, stream);
  const int d = out_view->d;
  DecParams p{};
  p.codes = codes; p.shapes = cb->shapes; p.gains = cb->gains; p.S = cb->S; p.K = cb->K; p.G = out_view->G;
  p.n_stages = n_stages; p.M = out_view->hd / d; p.N = out_view->T * p.M; p.out = kv_out; p.dtype = out_view->dtype;
  p.stride_g = out_view->stride_g; p.stride_t = out_view->stride_t;
  p.row_begin = 0;
  // bandwidth path: full 256-row chunks (d == 16, 1..4 stages, 16-byte aligned code planes)
  if (d == 16 && n_stages >= 1 && n_stages <= kDecDeep && p.N % 16 == 0 && p.N >= 256 && ((uintptr_t)codes & 15) == 0) {
    const long long n_chunks = p.N / 256;
    const bool dense = out_view->stride_t == out_view->hd;
    const int n_sm = sm_count();
    const bool deep = n_stages > 4;  // single-copy tables
    const size_t smem = deep ? (size_t)n_stages * (kDecTabBytes / 2) : (size_t)n_stages * kDecTabBytes;
    int per_sm = (int)((227 * 1024) / (smem + 1024));  // CTAs that fit on one SM (shared memory; 40 registers x 512 threads)
    if (per_sm > 2) per_sm = 2;  // measured: a third CTA per SM lowers the achieved bandwidth
    if (per_sm < 1) per_sm = 1;
    long long ctas = (per_sm * n_sm + out_view->G - 1) / out_view->G;
    const long long need = (n_chunks + kDecThreads / 32 - 1) / (kDecThreads / 32);
    if (ctas > need) ctas = need;
    dim3 grid((unsigned)ctas, (unsigned)out_view->G);
    // output addressing: dense rows, or a (head, token) slice of 8 rows = 128 contiguous elements (head_dim 128), or anything else
    const int layout = dense ? 1 : ((p.M == 8 && out_view->stride_t % 4 == 0) ? 2 : 0);
    const bool bf16 = out_view->dtype == GSRQ_BF16;
#define GSRQ_DEC_LAUNCH(NS, LAY, BF, DUPF)                                                                                          \
  do {                                                                                                                              \
    GSRQ_CUDA_CHECK(cudaFuncSetAttribute(k_decode_fast<NS, LAY, BF, DUPF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
    LAUNCH(kClsDecode, stream, (k_decode_fast<NS, LAY, BF, DUPF><<<grid, kDecThreads, smem, stream>>>(p, n_chunks)));                \
  } while (0)
#define GSRQ_DEC_FAST(NS, DUPF)                                                                 \
  do {                                                                                          \
    if (layout == 1) { if (bf16) GSRQ_DEC_LAUNCH(NS, 1, true, DUPF); else GSRQ_DEC_LAUNCH(NS, 1, false, DUPF); }      \
    else if (layout == 2) { if (bf16) GSRQ_DEC_LAUNCH(NS, 2, true, DUPF); else GSRQ_DEC_LAUNCH(NS, 2, false, DUPF); } \
    else { if (bf16) GSRQ_DEC_LAUNCH(NS, 0, true, DUPF); else GSRQ_DEC_LAUNCH(NS, 0, false, DUPF); }                  \
  } while (0)
    if (deep) GSRQ_DEC_FAST(kDecDeep, false);
    else if (n_stages == 1) GSRQ_DEC_FAST(1, true);
    else if (n_stages == 2) GSRQ_DEC_FAST(2, true);
    else if (n_stages == 3) GSRQ_DEC_FAST(3, true);
    else GSRQ_DEC_FAST(4, true);
#undef GSRQ_DEC_LAUNCH
#undef GSRQ_DEC_FAST
    GSRQ_CUDA_CHECK(cudaGetLastError());
    p.row_begin = n_chunks * 256;
    if (p.row_begin == p.N) return GSRQ_OK;
  }
  const size_t smem = (size_t)n_stages * cb->K * d * sizeof(float);
  const bool use_smem = smem <= 200 * 1024;
  // enough CTAs to fill the machine a few times, but few enough that the table load amortises
  const long long n_rows = p.N - p.row_begin;
  long long rows_per_cta = 8192;
  while (rows_per_cta > 1024 && (n_rows + rows_per_cta - 1) / rows_per_cta * out_view->G < 4 * 148) rows_per_cta /= 2;
  p.rows_per_cta = rows_per_cta;
  dim3 grid((unsigned)((n_rows + rows_per_cta - 1) / rows_per_cta), (unsigned)out_view->G);
  if (use_smem) {
    DISPATCH_D(d, {
      GSRQ_CUDA_CHECK(cudaFuncSetAttribute(k_decode<D, true, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(200 * 1024)));
      LAUNCH(kClsDecode, stream, (k_decode<D, true, 4><<<grid, 256, smem, stream>>>(p)));
    });
  } else {
    LAUNCH(kClsDecode, stream, DISPATCH_D(d, (k_decode<D, false, 4><<<grid, 256, 0, stream>>>(p))));
  }
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

int gsrq_encode_append(const void *kv_new, const gsrq_view *new_view, const gsrq_codebook *cb, int n_stages, uint8_t *codes,
                       int64_t plane_rows, int64_t t0, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!kv_new || !cb || !cb->shapes || !cb->gains || !codes) { set_error("NULL kv / codebook / codes"); return GSRQ_EINVAL; }
  int rc = check_view(new_view, cb->K, cb->S);
  if (rc) return rc;
  if (is_wide(new_view->d)) { set_error("gsrq_encode_append: d = %d is not supported (use gsrq_encode)", new_view->d); return GSRQ_EUNSUPPORTED; }
  const int M = new_view->hd / new_view->d;
  if (n_stages < 1 || n_stages > cb->S) { set_error("n_stages %d out of [1, %d]", n_stages, cb->S); return GSRQ_EINVAL; }
  if ((rc = check_align16(kv_new, "kv_new"))) return rc;
  if (t0 < 0 || plane_rows < (t0 + new_view->T) * M) { set_error("tokens [%lld, %lld) do not fit in planes of %lld rows", (long long)t0, (long long)(t0 + new_view->T), (long long)plane_rows); return GSRQ_EINVAL; }
  AppendParams p{};
  p.src = make_src(kv_new, new_view, nullptr, 0);
  p.N = new_view->T * M; p.shapes = cb->shapes; p.gains = cb->gains; p.S = cb->S; p.K = cb->K; p.n_stages = n_stages; p.G = new_view->G;
  p.codes = codes; p.code_stride_s = (long long)new_view->G * plane_rows; p.plane_rows = plane_rows; p.row0 = t0 * M;
  const long long rows = (long long)new_view->G * p.N;
  long long ctas = (rows + 7) / 8;
  if (ctas > 1184) ctas = 1184;
  const int d = new_view->d;
  LAUNCH(kClsEncode, stream, DISPATCH_D(d, (k_encode_append<D><<<(unsigned)ctas, 256, 0, stream>>>(p))));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

static int assign_all_rows(const void *kv, const gsrq_view *view, const float *residual, const gsrq_codebook *cb, int stage,
                           int mode, uint8_t *idx_out, float *dbg, void *workspace, size_t workspace_bytes, cudaStream_t stream) {
  if ((!kv && !residual) || !cb || !cb->shapes || !cb->gains || !idx_out) { set_error("NULL input"); return GSRQ_EINVAL; }
  int rc = check_view(view, cb->K, cb->S);
  if (rc) return rc;
  if (stage < 0 || stage >= cb->S || (mode != 0 && mode != 1)) { set_error("bad stage / mode"); return GSRQ_EINVAL; }
  if ((rc = check_align16(kv, "kv")) || (rc = check_align16(residual, "residual"))) return rc;
  if (is_wide(view->d)) {
    const WPlan wp = make_wplan(view, 0);
    rc = check_ws(workspace, workspace_bytes, wp.total);
    if (rc) return rc;
    char *wsw = (char *)workspace;
    const bool filter = wide_tc(view->d);
    if (dbg && !filter) { set_error("score dump needs the tensor-core path (d == 16, 64, 128)"); return GSRQ_EUNSUPPORTED; }
    const int n_planes = (!residual && view->dtype == GSRQ_BF16) ? 1 : 2;
    float *Rf = (float *)(wsw + wp.off_rows);
    rc = wide_prep(wp, view, make_src(kv, view, residual, wp.Nall), nullptr, 0, nullptr, view->T, wsw, filter, n_planes == 2, false, Rf, stream);
    if (rc) return rc;
    return wide_assign(wp, view, wsw, Rf, wp.Nall, cb->shapes + (size_t)stage * cb->K * view->d, cb->gains + (size_t)stage * cb->K, (long long)cb->S * cb->K,
                       cb->K, mode == 1 ? wide::kModeProj : wide::kModeGskm, filter, n_planes, idx_out, nullptr, 0, (unsigned int *)(wsw + wp.off_cnt), dbg, stream);
  }
  const Plan pl = make_plan(view, cb->K, cb->S, 0);
  rc = check_ws(workspace, workspace_bytes, pl.total);
  if (rc) return rc;
  char *ws = (char *)workspace;
  unsigned int *cnt = (unsigned int *)(ws + pl.off_cnt);
  GSRQ_CUDA_CHECK(cudaMemsetAsync(cnt, 0, sizeof(unsigned int), stream));
  const float *shapes_st = cb->shapes + (size_t)stage * cb->K * view->d;
  const float *gains_st = cb->gains + (size_t)stage * cb->K;
  if (use_tc(view->d)) {
    const int n_planes = (!residual && view->dtype == GSRQ_BF16) ? 1 : 2;
    rc = prepare_rows(pl, kv, view, nullptr, 0, nullptr, cb, 0, residual, ws, stream, n_planes);
    if (rc) return rc;
    const long long cb_stride_g = (long long)cb->S * cb->K;
    int *gmax = (int *)(ws + pl.off_gmax);
    LAUNCH(kClsMisc, stream, (tc::k_bimg<<<view->G, 256, 0, stream>>>(shapes_st, gains_st, cb_stride_g, 1, cb->K, mode,
                                                                      (uint8_t *)(ws + pl.off_bimg), gmax)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    TcMaps maps;
    rc = make_tc_maps(&maps, pl, ws, view->G, n_planes);
    if (rc) return rc;
    return run_assign_tc(pl, ws, maps, view->G, shapes_st, gains_st, cb_stride_g, cb->K, mode, n_planes, idx_out, nullptr, 0, gmax, 1,
                         dbg, stream);
  }
  if (dbg) { set_error("score dump needs the tensor-core path (d == 16)"); return GSRQ_EUNSUPPORTED; }
  EncParams p{};
  p.src = make_src(kv, view, residual, pl.Nall);
  p.N = pl.Nall; p.S = cb->S; p.K = cb->K;
  p.shapes = shapes_st; p.gains = gains_st;
  p.s_begin = 0; p.s_end = 1; p.s_base = 0; p.mode = mode; p.subtract = 0;
  p.codes = idx_out; p.code_stride_s = 0; p.res_out = nullptr; p.st = nullptr; p.slot = 0;
  p.list = (uint2 *)(ws + pl.off_list); p.list_cnt = cnt;
  return run_encode(p, view->G, view->d, stream);
}

int gsrq_assign(const void *kv, const gsrq_view *view, const float *residual, const gsrq_codebook *cb, int stage, int mode,
                uint8_t *idx_out, void *workspace, size_t workspace_bytes, gsrq_stream_t stream_) {
  return assign_all_rows(kv, view, residual, cb, stage, mode, idx_out, nullptr, workspace, workspace_bytes, (cudaStream_t)stream_);
}

int gsrq_debug_scores(const void *kv, const gsrq_view *view, const float *residual, const gsrq_codebook *cb, int stage, int mode,
                      float *scores_out, uint8_t *idx_out, void *workspace, size_t workspace_bytes, gsrq_stream_t stream_) {
  if (!scores_out) { set_error("NULL scores_out"); return GSRQ_EINVAL; }
  return assign_all_rows(kv, view, residual, cb, stage, mode, idx_out, scores_out, workspace, workspace_bytes, (cudaStream_t)stream_);
}

int gsrq_update(const void *kv, const gsrq_view *view, const float *residual, const float *w, int64_t w_stride_g,
                const uint8_t *idx, gsrq_codebook *cb, int stage, int shapes_too, void *workspace, size_t workspace_bytes,
                gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if ((!kv && !residual) || !cb || !cb->shapes || !cb->gains || !idx) { set_error("NULL input"); return GSRQ_EINVAL; }
  int rc = check_view(view, cb->K, cb->S);
  if (rc) return rc;
  if (stage < 0 || stage >= cb->S) { set_error("bad stage"); return GSRQ_EINVAL; }
  if (is_wide(view->d)) {
    const WPlan wp = make_wplan(view, 0);
    rc = check_ws(workspace, workspace_bytes, wp.total);
    if (rc) return rc;
    char *wsw = (char *)workspace;
    float *Rf = (float *)(wsw + wp.off_rows);
    rc = wide_prep(wp, view, make_src(kv, view, residual, wp.Nall), w, w_stride_g, nullptr, view->T, wsw, false, false, false, Rf, stream);
    if (rc) return rc;
    return wide_update(wp, view, wsw, Rf, wp.Nall, view->T, idx, cb->shapes + (size_t)stage * cb->K * view->d, cb->gains + (size_t)stage * cb->K,
                       (long long)cb->S * cb->K, cb->K, shapes_too ? 1 : 0, nullptr, 1, stream);
  }
  const Plan pl = make_plan(view, cb->K, cb->S, 0);
  rc = check_ws(workspace, workspace_bytes, pl.total);
  if (rc) return rc;
  char *ws = (char *)workspace;
  DevStats *st = (DevStats *)(ws + pl.off_st);
  GSRQ_CUDA_CHECK(cudaMemsetAsync(st, 0, (size_t)view->G * sizeof(DevStats), stream));
  // rows = residual when given, else kv as is (the caller states which stage's rows these are)
  rc = prepare_rows(pl, kv, view, w, w_stride_g, nullptr, cb, 0, residual, ws, stream);
  if (rc) return rc;
  if (use_tc(view->d))  // the fit's own reduction / merge phases (k_fit_tc.cuh), fed with the given assignment; rows from the fp32 buffer
    return run_fit_tc(pl, ws, nullptr, view->G, pl.M, cb->shapes + (size_t)stage * cb->K * view->d, cb->gains + (size_t)stage * cb->K,
                      (long long)cb->S * cb->K, cb->K, 2, const_cast<uint8_t *>(idx), nullptr, 1, 1, true, shapes_too ? 1 : 0, false, stream);
  return run_update(pl, view, cb->K, ws, idx, cb->shapes + (size_t)stage * cb->K * view->d,
                    cb->gains + (size_t)stage * cb->K, (long long)cb->S * cb->K, nullptr, shapes_too ? 1 : 0, 1, false, stream);
}

int gsrq_init_ids(const void *kv, const gsrq_view *view, const float *residual, const int64_t *fit_tokens, int64_t n_fit,
                  int K, int stage, uint64_t seed, int64_t *ids_out, void *workspace, size_t workspace_bytes, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if ((!kv && !residual) || !ids_out) { set_error("NULL input"); return GSRQ_EINVAL; }
  int rc = check_view(view, K, 1);
  if (rc) return rc;
  if (fit_tokens && (n_fit <= 0 || n_fit > view->T)) { set_error("n_fit out of range"); return GSRQ_EINVAL; }
  if (is_wide(view->d)) {
    const WPlan wp = make_wplan(view, fit_tokens ? n_fit : 0);
    if (wp.Nf < K) { set_error("fewer fit rows than codewords"); return GSRQ_EDEGENERATE; }
    rc = check_ws(workspace, workspace_bytes, wp.total);
    if (rc) return rc;
    char *wsw = (char *)workspace;
    DevStats *stw = (DevStats *)(wsw + wp.off_st);
    GSRQ_CUDA_CHECK(cudaMemsetAsync(stw, 0, (size_t)view->G * sizeof(DevStats), stream));
    float *Rf = (float *)(wsw + wp.off_rows);
    rc = wide_prep(wp, view, make_src(kv, view, residual, wp.Nall), nullptr, 0, (const long long *)fit_tokens, wp.nf_tok, wsw, false, false, false, Rf, stream);
    if (rc) return rc;
    LAUNCH(kClsPrep, stream, (wide::k_wide_init<<<view->G, 512, (size_t)K * sizeof(long long), stream>>>(Rf, wp.Nf, view->d, K, view->G, stage, seed, (long long *)ids_out, stw,
                                                                                                      nullptr, nullptr, 0, 0)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    return GSRQ_OK;
  }
  const Plan pl = make_plan(view, K, 1, fit_tokens ? n_fit : 0);
  if (pl.Nf < K) { set_error("fewer fit rows than codewords"); return GSRQ_EDEGENERATE; }
  rc = check_ws(workspace, workspace_bytes, pl.total);
  if (rc) return rc;
  char *ws = (char *)workspace;
  DevStats *st = (DevStats *)(ws + pl.off_st);
  GSRQ_CUDA_CHECK(cudaMemsetAsync(st, 0, (size_t)view->G * sizeof(DevStats), stream));
  rc = prepare_rows(pl, kv, view, nullptr, 0, (const long long *)fit_tokens, nullptr, 0, residual, ws, stream);
  if (rc) return rc;
  const int d = view->d;
  LAUNCH(kClsPrep, stream, DISPATCH_D(d, (k_init_ids<D><<<view->G, 512, 0, stream>>>((const float *)(ws + pl.off_Rf), pl.Nf, K, view->G,
                                                                                     stage, seed, (long long *)ids_out, st, nullptr,
                                                                                     nullptr, 0, nullptr))));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}


size_t gsrq_cluster_workspace_bytes(int64_t N, int d, int K) {
  if (check_cluster(N, d, K) != GSRQ_OK) return 0;
  return make_cplan(N, d, K).total;
}

int gsrq_cluster_fit(const float *x, const float *w, int64_t N, int d, int K, int iters, uint64_t seed, int method, float *shapes, float *gains,
                     uint16_t *idx_out, gsrq_fit_stats *stats, void *workspace, size_t workspace_bytes, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!x || !shapes || !gains || !idx_out) { set_error("NULL input"); return GSRQ_EINVAL; }
  int rc = check_cluster(N, d, K);
  if (rc) return rc;
  if (method != 0 && method != 1) { set_error("method must be 0 (GSKM) or 1 (K-means)"); return GSRQ_EINVAL; }
  if (iters < 0 || iters > GSRQ_MAX_ITERS) { set_error("iters must be in [0, %d]", GSRQ_MAX_ITERS); return GSRQ_EINVAL; }
  if ((rc = check_align16(x, "x"))) return rc;
  if (N < K) { set_error("fewer rows (%lld) than centroids (%d)", (long long)N, K); return GSRQ_EDEGENERATE; }
  const CPlan pl = make_cplan(N, d, K);
  rc = check_ws(workspace, workspace_bytes, pl.total);
  if (rc) return rc;
  char *ws = (char *)workspace;
  DevStats *st = (DevStats *)(ws + pl.off_st);
  float *Rf = (float *)(ws + pl.off_rows);
  GSRQ_CUDA_CHECK(cudaMemsetAsync(st, 0, sizeof(DevStats), stream));
  GSRQ_CUDA_CHECK(cudaMemsetAsync(idx_out, 0, (size_t)N * sizeof(uint16_t), stream));
  wide::WPrepParams q{};
  q.src.kv = nullptr; q.src.rows = x; q.src.dtype = GSRQ_F32; q.src.M = 1; q.src.d = d; q.src.stride_g = 0; q.src.stride_t = 0; q.src.rows_per_group = N;
  q.w = w; q.w_stride_g = 0; q.fit_tokens = nullptr; q.nf_tok = N; q.Rf = Rf; q.wt = (float *)(ws + pl.off_wt); q.wn = (double *)(ws + pl.off_wn);
  q.rnorm = (float *)(ws + pl.off_rnorm); q.epart = (double *)(ws + pl.off_epart); q.ahi = nullptr; q.alo = nullptr;
  LAUNCH(kClsPrep, stream, (wide::k_wide_prep<<<dim3((unsigned)pl.nE, 1), 256, 0, stream>>>(q)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  LAUNCH(kClsPrep, stream, (wide::k_wide_init<<<1, 512, (size_t)K * sizeof(long long), stream>>>(Rf, N, d, K, 1, 0, seed, (long long *)(ws + pl.off_ids), st, shapes, gains,
                                                                                                (long long)K, method)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  wide::WUpdateParams u{};
  u.rows = Rf; u.wn = (const double *)(ws + pl.off_wn); u.wt = (const float *)(ws + pl.off_wt); u.nf_tok = N; u.M = 1; u.idx = idx_out; u.idx16 = 1;
  u.N = N; u.d = d; u.K = K; u.shapes = shapes; u.gains = gains; u.cb_stride_g = K; u.st = st; u.term = (double *)(ws + pl.off_term);
  u.term_stride = kTermStride; u.term_k = K; u.gmax = nullptr; u.nparts = (N >= 8192) ? kWideParts : 1; u.part = (double *)(ws + pl.off_part);
  for (int t = (method == 1 ? 1 : 0); t <= iters; ++t) {   // GSKM: t = 0 is Alg. 1 l.2 (gains under the max-projection assignment)
    const int mode = (method == 1) ? wide::kModeKm : (t == 0 ? wide::kModeProj : wide::kModeGskm);
    rc = cluster_assign(Rf, N, d, K, mode, shapes, gains, idx_out, st, t, stream);
    if (rc) return rc;
    u.mode = (method == 1) ? 2 : (t > 0 ? 1 : 0); u.t = t;
    const dim3 ugrid((unsigned)K, 1, (unsigned)u.nparts);
    if (d > 128) LAUNCH(kClsUpdate, stream, (wide::k_wide_update<2><<<ugrid, 256, wide::wide_update_smem(), stream>>>(u)));
    else LAUNCH(kClsUpdate, stream, (wide::k_wide_update<1><<<ugrid, 256, wide::wide_update_smem(), stream>>>(u)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    if (u.nparts > 1) {
      LAUNCH(kClsUpdate, stream, (wide::k_wide_update_finish<<<dim3((unsigned)K, 1), 256, 0, stream>>>(u)));
      GSRQ_CUDA_CHECK(cudaGetLastError());
    }
    LAUNCH(kClsMisc, stream, (wide::k_wide_converged<<<1, 32, 0, stream>>>(st, 1, t)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
  }
  if (!stats) return GSRQ_OK;
  LAUNCH(kClsMisc, stream, (k_finish<<<1, 160, 0, stream>>>(st, (const double *)(ws + pl.off_term), kTermStride, K, (const double *)(ws + pl.off_epart), (int)pl.nE, iters, K)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return copy_fit_stats(st, 1, stats, stream);
}

int gsrq_cluster_assign(const float *x, int64_t N, int d, int K, int method, const float *shapes, const float *gains, uint16_t *idx_out,
                        gsrq_stream_t stream_) {
  if (!x || !shapes || !gains || !idx_out) { set_error("NULL input"); return GSRQ_EINVAL; }
  int rc = check_cluster(N, d, K);
  if (rc) return rc;
  if ((rc = check_align16(x, "x")) || (rc = check_align16(shapes, "shapes"))) return rc;
  return cluster_assign(x, N, d, K, method == 1 ? wide::kModeKm : wide::kModeGskm, shapes, gains, idx_out, nullptr, 0, (cudaStream_t)stream_);
}

int gsrq_cluster_metrics(const float *x, int64_t N, int d, int K, int method, const float *shapes, const float *gains, const uint16_t *idx,
                         double *out_host, void *workspace, size_t workspace_bytes, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!x || !shapes || !gains || !idx || !out_host) { set_error("NULL input"); return GSRQ_EINVAL; }
  int rc = check_cluster(N, d, K);
  if (rc) return rc;
  const CPlan pl = make_cplan(N, d, K);
  rc = check_ws(workspace, workspace_bytes, pl.total);
  if (rc) return rc;
  double *part = (double *)((char *)workspace + pl.off_met);
  double *res = part + (size_t)pl.nE * 5;
  LAUNCH(kClsMisc, stream, (wide::k_cluster_metrics<<<(unsigned)pl.nE, 256, 0, stream>>>(x, N, d, shapes, gains, idx, method == 1, K, part)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  LAUNCH(kClsMisc, stream, (wide::k_cluster_metrics_finish<<<1, 160, 0, stream>>>(part, pl.nE, N, res)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  GSRQ_CUDA_CHECK(cudaMemcpyAsync(out_host, res, 4 * sizeof(double), cudaMemcpyDeviceToHost, stream));
  GSRQ_CUDA_CHECK(cudaStreamSynchronize(stream));
  return GSRQ_OK;
}

static int attn_splits(int B, int G, long long max_len) {
  long long want = 4LL * sm_count() / ((long long)B * G);   // two CTAs fit on an SM: at most two full waves, no partial third one
  const long long cap = (max_len + 2047) / 2048;   // at least 2048 tokens per split: the per-CTA tables have to amortise
  if (want > cap) want = cap;
  if (want < 1) want = 1;
  if (want > 256) want = 256;
  return (int)want;
}

// d = 128: the dequantising kernel has no per-CTA table to amortise, so a split may be as short as 64 tokens (never fewer splits
// than attn_splits gives: the workspace is sized for this count).
static int attn_splits_wide(int B, int G, long long max_len) {
  long long want = 4LL * sm_count() / ((long long)B * G);
  const long long cap = (max_len + 63) / 64;
  if (want > cap) want = cap;
  if (want < 1) want = 1;
  if (want > 256) want = 256;
  return (int)want;
}

size_t gsrq_attention_workspace_bytes(int B, int Hq, int G, int64_t max_len) {
  if (B <= 0 || G <= 0 || Hq <= 0 || Hq % G || Hq / G > 8 || max_len < 0) { set_error("attention: bad B / Hq / G / max_len"); return 0; }
  return align_up((size_t)B * G * attn_splits_wide(B, G, max_len) * (Hq / G) * attn::kPartStride * sizeof(float)) + 256;
}

int gsrq_attention_decode(const float *q, const uint8_t *k_codes, const gsrq_codebook *k_cb, int k_stages, const uint8_t *v_codes,
                          const gsrq_codebook *v_cb, int v_stages, int64_t plane_rows, const int64_t *seq_start, const int64_t *seq_len,
                          int64_t max_len, int B, int Hq, int G, int hd, int d, float scale, float rope_theta, float *out, void *workspace,
                          size_t workspace_bytes, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!q || !k_codes || !v_codes || !k_cb || !v_cb || !k_cb->shapes || !k_cb->gains || !v_cb->shapes || !v_cb->gains || !seq_start || !seq_len || !out) {
    set_error("NULL input"); return GSRQ_EINVAL;
  }
  const bool wide_pt = (hd == attn::kHd && d == attn::kHd);   // the paper's operating point: one 128-wide sub-vector per token and head
  if (hd != attn::kHd || (d != attn::kD && !wide_pt)) { set_error("attention: this build serves head_dim 128 with d = 16 or d = 128 (got %d, %d)", hd, d); return GSRQ_EUNSUPPORTED; }
  const int max_stages = wide_pt ? GSRQ_MAX_STAGES : 4, rows_per_tok = wide_pt ? 1 : attn::kM;
  if (B <= 0 || G <= 0 || Hq <= 0 || Hq % G || Hq / G > 8) { set_error("attention: need Hq a multiple of G with at most 8 query heads per KV head"); return GSRQ_EINVAL; }
  if (B > 65535 || G > 65535) { set_error("attention: at most 65535 sequences and KV heads per call (grid limits), got B = %d, G = %d", B, G); return GSRQ_EINVAL; }
  if (((uintptr_t)k_cb->shapes & 15) || ((uintptr_t)v_cb->shapes & 15)) { set_error("codebook shapes must be 16-byte aligned"); return GSRQ_EINVAL; }
  if (k_cb->K < 1 || k_cb->K > 256 || v_cb->K < 1 || v_cb->K > 256 || k_stages < 1 || k_stages > max_stages || k_stages > k_cb->S || v_stages < 1 ||
      v_stages > max_stages || v_stages > v_cb->S) {
    set_error("attention: K in [1, 256] and 1..%d stages (<= S) for keys and values at d = %d", max_stages, d); return GSRQ_EINVAL;
  }
  if (plane_rows <= 0 || plane_rows % rows_per_tok || max_len < 0 || rope_theta < 0.0f) { set_error("attention: bad plane_rows / max_len / rope_theta"); return GSRQ_EINVAL; }
  if (!wide_pt && (((uintptr_t)k_codes & 7) || ((uintptr_t)v_codes & 7))) { set_error("code planes must be 8-byte aligned"); return GSRQ_EINVAL; }
  if ((uintptr_t)q & 15) { set_error("q must be 16-byte aligned"); return GSRQ_EINVAL; }
  const size_t need = gsrq_attention_workspace_bytes(B, Hq, G, max_len);
  int rc = check_ws(workspace, workspace_bytes, need);
  if (rc) return rc;
  attn::AttnParams p{};
  p.q = q; p.kc = k_codes; p.vc = v_codes; p.k_shapes = k_cb->shapes; p.k_gains = k_cb->gains; p.v_shapes = v_cb->shapes; p.v_gains = v_cb->gains;
  p.kS = k_cb->S; p.kK = k_cb->K; p.vS = v_cb->S; p.vK = v_cb->K; p.k_stages = k_stages; p.v_stages = v_stages; p.plane_rows = plane_rows;
  p.seq_start = (const long long *)seq_start; p.seq_len = (const long long *)seq_len; p.B = B; p.Hq = Hq; p.G = G; p.n_rep = Hq / G;
  p.n_split = wide_pt ? attn_splits_wide(B, G, max_len) : attn_splits(B, G, max_len);
  p.scale = scale; p.rope_theta = rope_theta; p.part = (float *)workspace; p.out = out;
  const bool rope = rope_theta > 0.0f;
  if (wide_pt) {   // d = 128: dequantising kernel (codeword rows from L2), then the same merge of the splits
    const dim3 wgrid((unsigned)p.n_split, (unsigned)G, (unsigned)B);
    if (rope) LAUNCH(kClsDecode, stream, (attn::k_attn_decode_wide<true><<<wgrid, attn::kThreads, 0, stream>>>(p)));
    else LAUNCH(kClsDecode, stream, (attn::k_attn_decode_wide<false><<<wgrid, attn::kThreads, 0, stream>>>(p)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    LAUNCH(kClsDecode, stream, (attn::k_attn_combine<<<dim3((unsigned)Hq, (unsigned)B), 128, 0, stream>>>(p)));
    GSRQ_CUDA_CHECK(cudaGetLastError());
    return GSRQ_OK;
  }
  const size_t smem = attn::attn_smem_bytes(k_stages, v_stages, p.n_rep, rope);
  if (smem > 227 * 1024) { set_error("attention: %d key stages x %d query heads per KV head do not fit in shared memory", k_stages, p.n_rep); return GSRQ_EUNSUPPORTED; }
  const dim3 grid((unsigned)p.n_split, (unsigned)G, (unsigned)B);
#define GSRQ_ATTN_K(KERNEL)                                                                                            \
  do {                                                                                                                \
    GSRQ_CUDA_CHECK(cudaFuncSetAttribute(KERNEL, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));            \
    LAUNCH(kClsDecode, stream, (KERNEL<<<grid, attn::kThreads, smem, stream>>>(p)));                                  \
  } while (0)
#define GSRQ_ATTN(NREP, NS)                                                                                           \
  do {                                                                                                                \
    if (rope) GSRQ_ATTN_K((attn::k_attn_decode_rope<NREP, NS>)); else GSRQ_ATTN_K((attn::k_attn_decode<false, NREP, NS>)); \
  } while (0)
  // compile-time head ratio / stage count for the common shapes (LLaMA-3-8B: 4 query heads per KV head); else the generic kernel
  const int ns = (k_stages == v_stages) ? k_stages : 0;
  if (p.n_rep == 4 && ns == 1) GSRQ_ATTN(4, 1);
  else if (p.n_rep == 4 && ns == 2) GSRQ_ATTN(4, 2);
  else if (p.n_rep == 4 && ns == 4) GSRQ_ATTN(4, 4);
  else if (p.n_rep == 1 && ns == 2) GSRQ_ATTN(1, 2);
  else if (p.n_rep == 8 && ns == 2) GSRQ_ATTN(8, 2);
  else GSRQ_ATTN(0, 0);
#undef GSRQ_ATTN_K
#undef GSRQ_ATTN
  GSRQ_CUDA_CHECK(cudaGetLastError());
  LAUNCH(kClsDecode, stream, (attn::k_attn_combine<<<dim3((unsigned)Hq, (unsigned)B), 128, 0, stream>>>(p)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

// ---- gsrq_attention_decode_static: the attention step for callers that have no way to hand over scratch memory ----
//
// The attention kernels leave one partial result (running max, sum, 128 accumulators) per (sequence, KV head, split, query head) in
// global memory and a second kernel merges the splits.  gsrq_attention_decode takes that buffer from the caller's workspace.  Here
// it lives in the library image instead: a fixed array in device global memory that the CUDA runtime places when it loads this
// module on a GPU, and that stays there until the process exits (every GPU this library is used on pays the 4 MiB once).
//
// g_attn_static_part, as host code sees it, is only a handle for the runtime; it is NOT the array's device address and must never
// be given to a kernel.  The address is asked for once per device (cudaGetSymbolAddress, with that device current) and kept in
// g_attn_static_ptr[device].
static __device__ __align__(256) float g_attn_static_part[GSRQ_ATTENTION_STATIC_SCRATCH_BYTES / sizeof(float)];
static float *g_attn_static_ptr[64] = {nullptr};
static std::mutex g_attn_static_mu;

// Device address of the static partial buffer on the CURRENT device (set-up on the first call per device, then a table lookup).
static int attn_static_scratch(float **out) {
  int dev = 0;
  GSRQ_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) { set_error("attention (static scratch): device ordinal %d out of range", dev); return GSRQ_ECUDA; }
  std::lock_guard<std::mutex> lk(g_attn_static_mu);
  if (!g_attn_static_ptr[dev]) {
    float *ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_attn_static_part);
    if (e != cudaSuccess || !ptr) {
      set_error("attention (static scratch): cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
      return GSRQ_ECUDA;
    }
    g_attn_static_ptr[dev] = ptr;
  }
  *out = g_attn_static_ptr[dev];
  return GSRQ_OK;
}

size_t gsrq_attention_static_scratch_bytes(void) { return sizeof(g_attn_static_part); }

int gsrq_attention_decode_static(const float *q, const uint8_t *k_codes, const gsrq_codebook *k_cb, int k_stages, const uint8_t *v_codes,
                                 const gsrq_codebook *v_cb, int v_stages, int64_t plane_rows, const int64_t *seq_start,
                                 const int64_t *seq_len, int64_t max_len, int B, int Hq, int G, int hd, int d, float scale,
                                 float rope_theta, float *out, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!q || !k_codes || !v_codes || !k_cb || !v_cb || !k_cb->shapes || !k_cb->gains || !v_cb->shapes || !v_cb->gains || !seq_start || !seq_len || !out) {
    set_error("NULL input"); return GSRQ_EINVAL;
  }
  if (hd != attn::kHd || d != attn::kD) { set_error("attention: this build serves head_dim 128 with d = 16 (got %d, %d)", hd, d); return GSRQ_EUNSUPPORTED; }
  if (B <= 0 || B > 65535 || G <= 0 || G > 65535 || Hq <= 0 || Hq % G || Hq / G > 8) {
    set_error("attention: need B, G <= 65535 and Hq a multiple of G with at most 8 query heads per KV head"); return GSRQ_EINVAL;
  }
  if (k_cb->K < 1 || k_cb->K > 256 || v_cb->K < 1 || v_cb->K > 256 || k_stages < 1 || k_stages > 4 || k_stages > k_cb->S || v_stages < 1 || v_stages > 4 ||
      v_stages > v_cb->S) { set_error("attention: K in [1, 256] and 1..4 stages (<= S) for keys and values"); return GSRQ_EINVAL; }
  if (plane_rows <= 0 || plane_rows % attn::kM || max_len < 0 || rope_theta < 0.0f) { set_error("attention: bad plane_rows / max_len / rope_theta"); return GSRQ_EINVAL; }
  if (((uintptr_t)k_codes & 7) || ((uintptr_t)v_codes & 7)) { set_error("code planes must be 8-byte aligned"); return GSRQ_EINVAL; }
  if (((uintptr_t)k_cb->shapes & 15) || ((uintptr_t)v_cb->shapes & 15)) { set_error("codebook shapes must be 16-byte aligned"); return GSRQ_EINVAL; }
  // the same split of the token range as gsrq_attention_decode (so the two paths add in the same order and agree bit for bit)
  const int n_split = attn_splits(B, G, max_len), n_rep = Hq / G;
  const size_t need = (size_t)B * G * n_split * n_rep * attn::kPartStride * sizeof(float);
  if (need > sizeof(g_attn_static_part)) {
    set_error("attention (static scratch): B = %d sequences x G = %d KV heads x %d splits x %d query heads per KV head need %zu bytes of "
              "partial results, the built-in buffer holds %zu; use gsrq_attention_decode with a workspace", B, G, n_split, n_rep, need,
              sizeof(g_attn_static_part));
    return GSRQ_EWORKSPACE;
  }
  float *part = nullptr;
  int rc = attn_static_scratch(&part);
  if (rc) return rc;
  attn::AttnParams p{};
  p.q = q; p.kc = k_codes; p.vc = v_codes; p.k_shapes = k_cb->shapes; p.k_gains = k_cb->gains; p.v_shapes = v_cb->shapes; p.v_gains = v_cb->gains;
  p.kS = k_cb->S; p.kK = k_cb->K; p.vS = v_cb->S; p.vK = v_cb->K; p.k_stages = k_stages; p.v_stages = v_stages; p.plane_rows = plane_rows;
  p.seq_start = (const long long *)seq_start; p.seq_len = (const long long *)seq_len; p.B = B; p.Hq = Hq; p.G = G; p.n_rep = n_rep;
  p.n_split = n_split; p.scale = scale; p.rope_theta = rope_theta; p.part = part; p.out = out;
  const bool rope = rope_theta > 0.0f;
  const size_t smem = attn::attn_smem_bytes(k_stages, v_stages, n_rep, rope);
  if (smem > 227 * 1024) { set_error("attention: %d key stages x %d query heads per KV head do not fit in shared memory", k_stages, n_rep); return GSRQ_EUNSUPPORTED; }
  const dim3 grid((unsigned)n_split, (unsigned)G, (unsigned)B);
  // Plain launches: no event pair around them even when gsrq_profile_enable is on (creating events is an allocation of its own).
  // Nothing in the buffer has to start at zero: every split's CTA stores all of its n_rep x 130 floats before the merge kernel,
  // which follows on the same stream, reads exactly the B x G x n_split x n_rep entries of THIS call.
#define GSRQ_ATTN_K(KERNEL)                                                                                            \
  do {                                                                                                                \
    GSRQ_CUDA_CHECK(cudaFuncSetAttribute(KERNEL, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));            \
    KERNEL<<<grid, attn::kThreads, smem, stream>>>(p);                                                                \
  } while (0)
#define GSRQ_ATTN(NREP, NS)                                                                                           \
  do {                                                                                                                \
    if (rope) GSRQ_ATTN_K((attn::k_attn_decode_rope<NREP, NS>)); else GSRQ_ATTN_K((attn::k_attn_decode<false, NREP, NS>)); \
  } while (0)
  const int ns = (k_stages == v_stages) ? k_stages : 0;
  if (n_rep == 4 && ns == 1) GSRQ_ATTN(4, 1);
  else if (n_rep == 4 && ns == 2) GSRQ_ATTN(4, 2);
  else if (n_rep == 4 && ns == 4) GSRQ_ATTN(4, 4);
  else if (n_rep == 1 && ns == 2) GSRQ_ATTN(1, 2);
  else if (n_rep == 8 && ns == 2) GSRQ_ATTN(8, 2);
  else GSRQ_ATTN(0, 0);
#undef GSRQ_ATTN_K
#undef GSRQ_ATTN
  GSRQ_CUDA_CHECK(cudaGetLastError());
  attn::k_attn_combine<<<dim3((unsigned)Hq, (unsigned)B), 128, 0, stream>>>(p);
  GSRQ_CUDA_CHECK(cudaGetLastError());
  {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    g_launches[kClsDecode] += 2;
  }
  return GSRQ_OK;
}

int gsrq_log_weights(const void *grad, const gsrq_view *view, float tau, float eps, float *w_out, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!grad || !view || !w_out) { set_error("NULL input"); return GSRQ_EINVAL; }
  if ((view->dtype != GSRQ_F32 && view->dtype != GSRQ_BF16) || view->G <= 0 || view->T <= 0 || view->hd <= 0) { set_error("bad view"); return GSRQ_EINVAL; }
  if (!(tau > 0.0f) || eps < 0.0f) { set_error("tau must be > 0 and eps >= 0"); return GSRQ_EINVAL; }
  dim3 grid((unsigned)((view->T + 7) / 8), (unsigned)view->G);
  LAUNCH(kClsPrep, stream, (var::k_grad_norms<<<grid, 256, 0, stream>>>(grad, view->dtype, view->hd, view->T, view->stride_g, view->stride_t, w_out)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  LAUNCH(kClsPrep, stream, (var::k_log_weights<<<view->G, 1024, 0, stream>>>(w_out, view->T, (double)tau, (double)eps)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

int gsrq_encode_pervector_gain(const void *kv, const gsrq_view *view, const gsrq_codebook *cb, int n_stages, uint8_t *codes, uint16_t *gains16,
                               float *residual, void *workspace, size_t workspace_bytes, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!kv || !cb || !cb->shapes || !cb->gains || !codes || !gains16 || !residual) { set_error("NULL input (the fp32 residual buffer is required)"); return GSRQ_EINVAL; }
  int rc = check_view(view, cb->K, cb->S);
  if (rc) return rc;
  if (is_wide(view->d)) { set_error("per-vector gain codes: d in {8, 16, 32}"); return GSRQ_EUNSUPPORTED; }
  if (n_stages < 1 || n_stages > cb->S) { set_error("n_stages %d out of [1, %d]", n_stages, cb->S); return GSRQ_EINVAL; }
  if ((rc = check_align16(kv, "kv")) || (rc = check_align16(residual, "residual"))) return rc;
  const int G = view->G, d = view->d, M = view->hd / d;
  const long long N = view->T * M;
  for (int s = 0; s < n_stages; ++s) {
    uint8_t *plane = codes + (size_t)s * G * N;
    // shape of the stage: arg-max of the plain projection r . s_k (exact, lowest index on ties)
    rc = gsrq_assign(kv, view, s ? residual : nullptr, cb, s, 1, plane, workspace, workspace_bytes, stream_);
    if (rc) return rc;
    var::PvgParams p{};
    p.src = make_src(kv, view, s ? residual : nullptr, N); p.N = N; p.shapes = cb->shapes + (size_t)s * cb->K * d; p.cb_stride_g = (long long)cb->S * cb->K;
    p.codes = plane; p.gains = reinterpret_cast<__half *>(gains16) + (size_t)s * G * N; p.res_out = residual;
    dim3 grid((unsigned)((N + 255) / 256), (unsigned)G);
    LAUNCH(kClsEncode, stream, DISPATCH_D(d, (var::k_pvg_finish<D><<<grid, 256, 0, stream>>>(p))));
    GSRQ_CUDA_CHECK(cudaGetLastError());
  }
  return GSRQ_OK;
}

int gsrq_decode_pervector_gain(const uint8_t *codes, const uint16_t *gains16, const gsrq_codebook *cb, int n_stages, void *kv_out,
                               const gsrq_view *out_view, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!codes || !gains16 || !cb || !cb->shapes || !kv_out) { set_error("NULL input"); return GSRQ_EINVAL; }
  int rc = check_view(out_view, cb->K, cb->S);
  if (rc) return rc;
  if (is_wide(out_view->d)) { set_error("per-vector gain codes: d in {8, 16, 32}"); return GSRQ_EUNSUPPORTED; }
  if (n_stages < 0 || n_stages > cb->S) { set_error("n_stages %d out of [0, %d]", n_stages, cb->S); return GSRQ_EINVAL; }
  var::PvgDecParams p{};
  p.codes = codes; p.gains = reinterpret_cast<const __half *>(gains16); p.shapes = cb->shapes; p.S = cb->S; p.K = cb->K; p.G = out_view->G;
  p.n_stages = n_stages; p.M = out_view->hd / out_view->d; p.N = out_view->T * p.M; p.out = kv_out; p.dtype = out_view->dtype;
  p.stride_g = out_view->stride_g; p.stride_t = out_view->stride_t;
  dim3 grid((unsigned)((p.N + 255) / 256), (unsigned)out_view->G);
  const int d = out_view->d;
  LAUNCH(kClsDecode, stream, DISPATCH_D(d, (var::k_pvg_decode<D><<<grid, 256, 0, stream>>>(p))));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

int gsrq_pack_nibbles(const uint8_t *codes, int K, int64_t n_planes, int64_t N, uint8_t *packed, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!codes || !packed || n_planes <= 0 || N <= 0) { set_error("bad arguments"); return GSRQ_EINVAL; }
  if (K < 1 || K > 16) { set_error("nibble packing holds codes of K <= 16 codewords, got K = %d", K); return GSRQ_EINVAL; }
  LAUNCH(kClsMisc, stream, (var::k_pack_nibbles<<<1184, 256, 0, stream>>>(codes, n_planes, N, packed)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

int gsrq_unpack_nibbles(const uint8_t *packed, int64_t n_planes, int64_t N, uint8_t *codes, gsrq_stream_t stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!codes || !packed || n_planes <= 0 || N <= 0) { set_error("bad arguments"); return GSRQ_EINVAL; }
  LAUNCH(kClsMisc, stream, (var::k_unpack_nibbles<<<1184, 256, 0, stream>>>(packed, n_planes, N, codes)));
  GSRQ_CUDA_CHECK(cudaGetLastError());
  return GSRQ_OK;
}

int gsrq_encode_host(const void *kv_host, const gsrq_view *view, const gsrq_codebook *cb, uint8_t *codes_host) {
  if (!kv_host || !cb || !codes_host) { set_error("NULL input"); return GSRQ_EINVAL; }
  int rc = check_view(view, cb->K, cb->S);
  if (rc) return rc;
  // host buffer must be one dense block covering the view
  const size_t esz = view->dtype == GSRQ_BF16 ? 2 : 4;
  const size_t n_el = (size_t)view->G * view->T * view->hd;
  const size_t n_codes = (size_t)cb->S * view->G * view->T * (view->hd / view->d);
  const size_t wsb = gsrq_workspace_bytes(view, cb->K, cb->S, 0);
  void *d_kv = nullptr, *d_codes = nullptr, *d_ws = nullptr;
  cudaStream_t stream = nullptr;
  cudaError_t e = cudaMalloc(&d_kv, n_el * esz);
  if (e == cudaSuccess) e = cudaMalloc(&d_codes, n_codes);
  if (e == cudaSuccess) e = cudaMalloc(&d_ws, wsb);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_kv, kv_host, n_el * esz, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess) {
    rc = gsrq_encode(d_kv, view, cb, 0, cb->S, (uint8_t *)d_codes, nullptr, d_ws, wsb, stream);
    if (rc == GSRQ_OK) e = cudaMemcpyAsync(codes_host, d_codes, n_codes, cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
  }
  cudaFree(d_kv); cudaFree(d_codes); cudaFree(d_ws);
  if (e != cudaSuccess) { set_error("gsrq_encode_host: %s", cudaGetErrorString(e)); return GSRQ_ECUDA; }
  return rc;
}

int gsrq_decode_host(const uint8_t *codes_host, const gsrq_codebook *cb, int n_stages, void *kv_out_host,
                     const gsrq_view *out_view) {
  if (!codes_host || !cb || !kv_out_host) { set_error("NULL input"); return GSRQ_EINVAL; }
  int rc = check_view(out_view, cb->K, cb->S);
  if (rc) return rc;
  const size_t esz = out_view->dtype == GSRQ_BF16 ? 2 : 4;
  const size_t n_el = (size_t)out_view->G * out_view->T * out_view->hd;
  const size_t n_codes = (size_t)cb->S * out_view->G * out_view->T * (out_view->hd / out_view->d);
  void *d_kv = nullptr, *d_codes = nullptr;
  cudaStream_t stream = nullptr;
  cudaError_t e = cudaMalloc(&d_kv, n_el * esz);
  if (e == cudaSuccess) e = cudaMalloc(&d_codes, n_codes);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_codes, codes_host, n_codes, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess) {
    rc = gsrq_decode((const uint8_t *)d_codes, cb, n_stages, d_kv, out_view, stream);
    if (rc == GSRQ_OK) e = cudaMemcpyAsync(kv_out_host, d_kv, n_el * esz, cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
  }
  cudaFree(d_kv); cudaFree(d_codes);
  if (e != cudaSuccess) { set_error("gsrq_decode_host: %s", cudaGetErrorString(e)); return GSRQ_ECUDA; }
  return rc;
}


// ---- the *_host entry points' private stream-ordered pool (one per device, kept between calls) ----
static std::mutex g_pool_mu;
static cudaMemPool_t g_pools[64] = {nullptr};

static cudaMemPool_t host_pool() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
  std::lock_guard<std::mutex> lk(g_pool_mu);
  if (!g_pools[dev]) {
    cudaMemPoolProps props;
    memset(&props, 0, sizeof(props));
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t pool = nullptr;
    if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    unsigned long long keep = ~0ull;   // keep the memory between calls (gsrq_release_host_pool() returns it)
    cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    g_pools[dev] = pool;
  }
  return g_pools[dev];
}

__global__ void k_collect_err(const DevStats *__restrict__ st, int G, int *__restrict__ err_accum) {
  for (int g = threadIdx.x; g < G; g += blockDim.x)
    if (st[g].err) atomicMin(err_accum, st[g].err);   // error codes are negative: keep the lowest
}

// One tensor's chain of the host pipeline, enqueued on `stream` (nothing here waits for the device).  h2d_after: the upload
// waits for this event (the previous tensor's upload, so that uploads run one after the other at full link speed instead of
// sharing it); h2d_done is recorded after this tensor's upload.
struct PipeJob {
  char *base = nullptr;
  cudaStream_t stream = nullptr;
  int *h_err = nullptr;   // pinned: a download into pageable memory would block the enqueueing thread until the chain is done
  int rc = GSRQ_OK;
  cudaError_t e = cudaSuccess;
};

static void pipeline_enqueue(PipeJob &jb, cudaMemPool_t pool, const void *kv_host, const gsrq_view *view, const float *w_host,
                             const int64_t *fit_tokens_host, int64_t n_fit, int K, int S, int iters, uint64_t seed, float *shapes_host,
                             float *gains_host, uint8_t *codes_host, void *kv_out_host, cudaEvent_t h2d_after, cudaEvent_t h2d_done) {
  const int G = view->G, d = view->d, M = view->hd / d;
  const size_t esz = view->dtype == GSRQ_BF16 ? 2 : 4;
  const size_t kv_bytes = (size_t)G * view->T * view->hd * esz;
  const size_t n_rows = (size_t)G * view->T * M;
  const size_t sh_bytes = (size_t)G * S * K * d * 4, ga_bytes = (size_t)G * S * K * 4;
  const size_t ft_bytes = fit_tokens_host ? (size_t)G * n_fit * sizeof(int64_t) : 0;
  const size_t wsb = gsrq_workspace_bytes(view, K, S, fit_tokens_host ? n_fit : 0);
  const bool per_stage = !fit_tokens_host;   // fit on all tokens: encode each stage after its fit, its residual feeds the next fit
  cudaStream_t stream = jb.stream;
  size_t off[10], o = 0;
  const size_t sizes[10] = {kv_bytes, (size_t)view->T * 4, sh_bytes, ga_bytes, n_rows * S, per_stage ? n_rows * d * 4 : 0, wsb,
                            kv_out_host ? kv_bytes : 0, ft_bytes, 256};
  for (int i = 0; i < 10; ++i) { off[i] = o; o += align_up(sizes[i]); }
  cudaError_t &e = jb.e;
  int &rc = jb.rc;
  e = cudaMallocFromPoolAsync((void **)&jb.base, o, pool, stream);
  if (e != cudaSuccess) { jb.base = nullptr; return; }
  char *base = jb.base;
  void *d_kv = base + off[0];
  float *d_w = w_host ? (float *)(base + off[1]) : nullptr;
  gsrq_codebook cb{K, S, (float *)(base + off[2]), (float *)(base + off[3])};
  uint8_t *d_codes = (uint8_t *)(base + off[4]);
  float *d_res = per_stage ? (float *)(base + off[5]) : nullptr;
  void *d_ws = base + off[6], *d_out = base + off[7];
  int64_t *d_ft = fit_tokens_host ? (int64_t *)(base + off[8]) : nullptr;
  int *d_err = (int *)(base + off[9]);
  const Plan pl = make_plan(view, K, S, fit_tokens_host ? n_fit : 0);
  if (h2d_after) e = cudaStreamWaitEvent(stream, h2d_after, 0);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_kv, kv_host, kv_bytes, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess && h2d_done) e = cudaEventRecord(h2d_done, stream);
  if (e == cudaSuccess && w_host) e = cudaMemcpyAsync(d_w, w_host, (size_t)view->T * 4, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess && d_ft) e = cudaMemcpyAsync(d_ft, fit_tokens_host, ft_bytes, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_err, 0, sizeof(int), stream);
  for (int s = 0; s < S && rc == GSRQ_OK && e == cudaSuccess; ++s) {
    rc = gsrq_fit_stage(d_kv, view, d_w, 0, d_ft, n_fit, &cb, s, (per_stage && s) ? d_res : nullptr, iters, seed, nullptr, d_ws, wsb, stream);
    if (rc == GSRQ_OK) {   // remember a failed initialisation (the stage's statistics are reset by the next fit)
      const size_t off_st = is_wide(d) ? make_wplan(view, fit_tokens_host ? n_fit : 0).off_st : pl.off_st;
      k_collect_err<<<1, 128, 0, stream>>>((const DevStats *)((char *)d_ws + off_st), G, d_err);
      e = cudaGetLastError();
    }
    if (per_stage && rc == GSRQ_OK && e == cudaSuccess) {
      // the fused tensor-core encode restarts from stage 0 (cheap); otherwise only stage s is encoded
      const int sb = can_encode_tc(d_kv, view, 0) ? 0 : s;
      rc = gsrq_encode(d_kv, view, &cb, sb, s + 1, d_codes, (s + 1 < S) ? d_res : nullptr, d_ws, wsb, stream);
    }
  }
  if (!per_stage && rc == GSRQ_OK && e == cudaSuccess) rc = gsrq_encode(d_kv, view, &cb, 0, S, d_codes, nullptr, d_ws, wsb, stream);
  if (rc == GSRQ_OK && e == cudaSuccess && kv_out_host) {
    rc = gsrq_decode(d_codes, &cb, S, d_out, view, stream);
    if (rc == GSRQ_OK) e = cudaMemcpyAsync(kv_out_host, d_out, kv_bytes, cudaMemcpyDeviceToHost, stream);
  }
  if (rc == GSRQ_OK && e == cudaSuccess) e = cudaMemcpyAsync(shapes_host, cb.shapes, sh_bytes, cudaMemcpyDeviceToHost, stream);
  if (rc == GSRQ_OK && e == cudaSuccess) e = cudaMemcpyAsync(gains_host, cb.gains, ga_bytes, cudaMemcpyDeviceToHost, stream);
  if (rc == GSRQ_OK && e == cudaSuccess) e = cudaMemcpyAsync(codes_host, d_codes, n_rows * S, cudaMemcpyDeviceToHost, stream);
  if (rc == GSRQ_OK && e == cudaSuccess) e = cudaMemcpyAsync(jb.h_err, d_err, sizeof(int), cudaMemcpyDeviceToHost, stream);
}

// Waits for the job's stream, returns its memory to the pool; the job's status.
static int pipeline_finish(PipeJob &jb) {
  if (jb.base) cudaFreeAsync(jb.base, jb.stream);
  const cudaError_t e2 = cudaStreamSynchronize(jb.stream);
  if (jb.e == cudaSuccess) jb.e = e2;
  if (jb.e != cudaSuccess) { set_error("gsrq_pipeline_host: %s", cudaGetErrorString(jb.e)); cudaGetLastError(); return GSRQ_ECUDA; }
  if (jb.rc == GSRQ_OK && *jb.h_err == GSRQ_EDEGENERATE) { set_error("a group has fewer than K distinct non-zero fit rows"); return GSRQ_EDEGENERATE; }
  if (jb.rc == GSRQ_OK && *jb.h_err != 0) { set_error("the fit kernel's group barrier timed out"); return GSRQ_ECUDA; }
  return jb.rc;
}

int gsrq_pipeline_host_batch(int n, const void *const *kv_host, const gsrq_view *view, const float *const *w_host,
                             const int64_t *const *fit_tokens_host, int64_t n_fit, int K, int S, int iters, uint64_t seed,
                             float *const *shapes_host, float *const *gains_host, uint8_t *const *codes_host, void *const *kv_out_host) {
  if (n <= 0 || n > 64 || !kv_host || !shapes_host || !gains_host || !codes_host) { set_error("gsrq_pipeline_host_batch: need 1..64 tensors and non-NULL pointer arrays"); return GSRQ_EINVAL; }
  int rc = check_view(view, K, S);
  if (rc) return rc;
  for (int i = 0; i < n; ++i) {
    if (!kv_host[i] || !shapes_host[i] || !gains_host[i] || !codes_host[i]) { set_error("NULL input (tensor %d)", i); return GSRQ_EINVAL; }
    const int64_t *ft = fit_tokens_host ? fit_tokens_host[i] : nullptr;
    if (ft && (n_fit <= 0 || n_fit > view->T)) { set_error("n_fit out of range"); return GSRQ_EINVAL; }
  }
  cudaMemPool_t pool = host_pool();
  if (!pool) { set_error("gsrq_pipeline_host: could not create the device memory pool"); return GSRQ_ECUDA; }
  // two streams, tensors alternate between them: tensor i + 1 uploads while tensor i computes and downloads (the two copy
  // directions and the SMs work at the same time); a stream's next tensor starts when its previous one is done
  cudaStream_t st[2] = {nullptr, nullptr};
  cudaEvent_t up[2] = {nullptr, nullptr};
  const int ns = n > 1 ? 2 : 1;
  cudaError_t e = cudaSuccess;
  for (int q = 0; q < ns && e == cudaSuccess; ++q) {
    e = cudaStreamCreateWithFlags(&st[q], cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&up[q], cudaEventDisableTiming);
  }
  std::vector<PipeJob> jobs((size_t)n);
  int first_bad = GSRQ_OK;
  int *h_errs = nullptr;
  if (e == cudaSuccess) e = cudaHostAlloc((void **)&h_errs, (size_t)n * sizeof(int), cudaHostAllocDefault);
  if (e == cudaSuccess) {
    for (int i = 0; i < n; ++i) {
      PipeJob &jb = jobs[(size_t)i];
      jb.stream = st[i % ns];
      jb.h_err = h_errs + i;
      *jb.h_err = 0;
      if (i >= ns) { const int r = pipeline_finish(jobs[(size_t)(i - ns)]); if (r != GSRQ_OK && first_bad == GSRQ_OK) first_bad = r; }   // its stream (and event) are free again
      pipeline_enqueue(jb, pool, kv_host[i], view, w_host ? w_host[i] : nullptr, fit_tokens_host ? fit_tokens_host[i] : nullptr, n_fit, K, S, iters, seed,
                       shapes_host[i], gains_host[i], codes_host[i], kv_out_host ? kv_out_host[i] : nullptr, (i > 0 && ns > 1) ? up[(i - 1) % ns] : nullptr,
                       ns > 1 ? up[i % ns] : nullptr);
    }
    for (int i = (n > ns ? n - ns : 0); i < n; ++i) { const int r = pipeline_finish(jobs[(size_t)i]); if (r != GSRQ_OK && first_bad == GSRQ_OK) first_bad = r; }
  }
  for (int q = 0; q < ns; ++q) { if (up[q]) cudaEventDestroy(up[q]); if (st[q]) cudaStreamDestroy(st[q]); }
  if (h_errs) cudaFreeHost(h_errs);
  if (e != cudaSuccess) { set_error("gsrq_pipeline_host: %s", cudaGetErrorString(e)); return GSRQ_ECUDA; }
  return first_bad;
}

int gsrq_pipeline_host(const void *kv_host, const gsrq_view *view, const float *w_host, const int64_t *fit_tokens_host,
                       int64_t n_fit, int K, int S, int iters, uint64_t seed, float *shapes_host, float *gains_host,
                       uint8_t *codes_host, void *kv_out_host) {
  if (!kv_host || !shapes_host || !gains_host || !codes_host) { set_error("NULL input"); return GSRQ_EINVAL; }
  return gsrq_pipeline_host_batch(1, &kv_host, view, &w_host, &fit_tokens_host, n_fit, K, S, iters, seed, &shapes_host, &gains_host, &codes_host,
                                  &kv_out_host);
}

void gsrq_release_host_pool(void) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return;
  std::lock_guard<std::mutex> lk(g_pool_mu);
  if (g_pools[dev]) { cudaMemPoolDestroy(g_pools[dev]); g_pools[dev] = nullptr; }
}

void gsrq_profile_enable(int on) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  g_prof_on = on != 0;
}

int gsrq_profile_read(double *ms_by_class, int64_t *launches_by_class) {
  std::vector<ProfRec> recs;
  {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    recs.swap(g_prof_recs);
  }
  for (int c = 0; c < kNumCls; ++c) { if (ms_by_class) ms_by_class[c] = 0.0; if (launches_by_class) launches_by_class[c] = 0; }
  int rc = GSRQ_OK;
  for (auto &r : recs) {
    float ms = 0.f;
    cudaError_t e = cudaEventSynchronize(r.b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, r.a, r.b);
    if (e != cudaSuccess) { set_error("profile read: %s", cudaGetErrorString(e)); rc = GSRQ_ECUDA; }
    else { if (ms_by_class) ms_by_class[r.cls] += ms; if (launches_by_class) launches_by_class[r.cls] += 1; }
    cudaEventDestroy(r.a); cudaEventDestroy(r.b);
  }
  return rc;
}

int64_t gsrq_launch_count(void) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  long long n = 0;
  for (int c = 0; c < kNumCls; ++c) n += g_launches[c];
  return n;
}

}  // extern "C"
