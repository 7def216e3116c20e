/*
 * gsrq.h -- C ABI of libgsrq: the GSRQ residual-quantization encoder (weighted
 * Gain-Shape K-means codebook fit + per-stage encode) and the stand-alone decode,
 * hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Citations are to the paper text, /root/reference/PAPER.md ("PAPER.md:<line>" plus
 * section / equation / algorithm), and to DESIGN.md for the readings taken where the
 * paper is silent.
 *
 * Conventions (all entry points)
 *   - Every pointer is a DEVICE pointer owned by the caller, except: the small structs
 *     (gsrq_view, gsrq_codebook -- host structs holding device pointers), `stats`
 *     (host), and the *_host entry points at the bottom, which say so.
 *   - The device entry points allocate nothing; scratch comes from the caller's `workspace`
 *     (>= gsrq_workspace_bytes(), 256-byte aligned).  Only the *_host entry points at the bottom
 *     allocate: from a private, library-owned stream-ordered memory pool that is kept between
 *     calls and released by gsrq_release_host_pool() (the process-wide default pool is not touched).
 *   - Tensor base pointers (kv, kv_out, residual, residual_out, kv_new) must be 16-byte aligned
 *     (vector loads / stores); a misaligned pointer returns GSRQ_EINVAL.
 *   - Calls are asynchronous on `stream`.  The only implied synchronisation is the
 *     copy of `stats` to the host in gsrq_fit_stage (skipped when stats == NULL).
 *   - Return value: GSRQ_OK (0) or a negative gsrq_status; never throws, never
 *     aborts.  After an error the outputs are unspecified; gsrq_last_error() returns a
 *     thread-local message.
 *   - Same inputs => bit-identical outputs on every run (no floating-point atomics).
 *   - There is no CPU fallback: without a CUDA device every compute entry point
 *     returns GSRQ_ECUDA.
 *
 * Notation: a KV tensor of G heads x T tokens x hd
 * channels is split into M = hd/d sub-vectors ("rows") of dimension d per (head,
 * token) (Product Quantization); row i = t*M + m of head g is kv[g][t][m*d..m*d+d).
 * Each head g and residual stage s has one codebook of K centroids
 * mu_k = g_k * s_k, g_k >= 0, ||s_k|| = 1 (Eq. 3).  A code is the index k (uint8).
 */
#ifndef GSRQ_H_
#define GSRQ_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GSRQ_MAX_ITERS 128 /* PAPER.md:479 "setting the maximum iteration to around 100 is sufficient" */
#define GSRQ_MAX_K 256     /* codes are one byte; PAPER.md:250 uses K = 256 throughout */
#define GSRQ_MAX_STAGES 32 /* PAPER.md:252 R = 32 for 2 BPA */

typedef enum {
  GSRQ_OK = 0,
  GSRQ_EINVAL = -1,       /* bad shape / alignment / K > 256 / hd % d != 0 / NULL pointer */
  GSRQ_EUNSUPPORTED = -2, /* valid request this build has no kernel for (d not in {8,16,32,64,128,256}) */
  GSRQ_EWORKSPACE = -3,   /* workspace too small or misaligned */
  GSRQ_ECUDA = -4,        /* CUDA runtime error (message in gsrq_last_error) */
  GSRQ_EDEGENERATE = -5   /* a group has fewer than K distinct non-zero fit rows (init impossible) */
} gsrq_status;

enum { GSRQ_F32 = 0, GSRQ_BF16 = 1 };

/* A CUDA stream (the same type as cudaStream_t / CUstream; declared here so that this header needs no CUDA header). */
typedef struct CUstream_st *gsrq_stream_t;

/* Strided view of one layer's K or V cache.  Innermost hd elements are contiguous.
 * [G][T][hd] -> stride_g = T*hd, stride_t = hd;  [T][G][hd] -> stride_g = hd, stride_t = G*hd. */
typedef struct {
  int32_t dtype;    /* GSRQ_F32 or GSRQ_BF16 */
  int32_t G;        /* codebook groups = KV heads */
  int64_t T;        /* tokens (batch folded in) */
  int32_t hd, d;    /* head_dim and sub-vector dim; hd % d == 0 */
  int64_t stride_g; /* in elements */
  int64_t stride_t; /* in elements */
} gsrq_view;

/* Codebooks of all stages (device arrays, caller-owned):
 * shapes [G][S][K][d] fp32 unit-norm, gains [G][S][K] fp32 >= 0  (Eq. 3). */
typedef struct {
  int32_t K, S;
  float *shapes;
  float *gains;
} gsrq_codebook;

/* Per-group statistics of one gsrq_fit_stage call (host struct; pass an array of G). */
typedef struct {
  int32_t iters_run;     /* Lloyd iterations executed before Alg. 1 l.15-16 broke (<= iters) */
  int32_t n_empty_last;  /* empty clusters at the last update (kept unchanged) */
  int64_t n_changed_last;
  int64_t n_refined;     /* rows whose arg-max went through the exact fp64 re-score */
  double wdist_after_assign[GSRQ_MAX_ITERS]; /* J_t = sum_i w_i ||r_i - g s||^2 after iteration t's assignment */
  int64_t n_changed[GSRQ_MAX_ITERS];         /* rows whose assignment changed at iteration t */
} gsrq_fit_stats;

/* Scratch size for any call on this view with these parameters.
 * n_fit_tokens > 0: size of the fit subset; 0: "fit on all T tokens"; < 0: no fit at all
 * (gsrq_encode / gsrq_decode only).  Host function, no CUDA calls. */
size_t gsrq_workspace_bytes(const gsrq_view *view, int K, int S, int64_t n_fit_tokens);

/*
 * Fit the codebook of residual stage `stage` with weighted GSKM.
 *   Algorithm 1 with per-sample weights (reading c-W):
 *   init: K seeded distinct non-zero fit rows, normalised (Alg. 1 l.1; reading c-I), gains by
 *   Eq. 8 under the max-projection assignment (l.2); then up to `iters` iterations of
 *   assignment  k_i = argmax_k (2 g_k r_i.s_k - g_k^2), lowest k on ties   (Eq. 5)
 *   update      s_k = normalize(sum w_i y_i), y_i = r_i/(||r_i|| + 1e-12)   (Eq. 6-7)
 *               g_k = max(0, sum w_i r_i.s_k / sum w_i) with the new s_k    (Eq. 8)
 *   with the safeguards of PAPER.md:178 (empty cluster and near-zero direction keep the old
 *   value) and the early exit of Alg. 1 l.15-16.
 * kv       : the tensor described by `view` (read-only).
 * w        : [.][T] fp32 per-token weights, row of group g at w + g*w_stride_g (0 = shared);
 *            NULL = uniform.  A sub-vector inherits its token's weight.
 * fit_tokens: [G][n_fit] int64 sorted token ids the codebook is fitted on; NULL = all T
 *            tokens (then n_fit is ignored).
 * cb       : stages < `stage` are read (only when residual == NULL and stage > 0),
 *            stage `stage` is written.
 * residual : [G][T*M][d] fp32 residual after stage-1 (gsrq_encode's residual_out), or NULL:
 *            stage 0 reads kv; stage > 0 re-derives the residual from kv and cb.
 * seed     : selects the initial rows (splitmix64 stream, reading c-I).
 * stats    : HOST array of G structs or NULL.  When given, the call synchronises `stream`
 *            and returns GSRQ_EDEGENERATE if any group could not be initialised; the per-iteration
 *            distortions are only computed in that case.  With stats == NULL the call is asynchronous and
 *            detection of those errors is deferred to gsrq_fit_status (below).
 * Kernels  : d == 16: ONE persistent cooperative kernel runs all passes (tcgen05 filter with an fp64 re-score of
 *            the ambiguous rows, per-CTA fp64 reduction, merge + Eq. 7-8, two group barriers per pass) and
 *            leaves the loop when a group's assignments stop changing (Alg. 1 l.15-16).  Other d: two
 *            launches per pass (CUDA-core filter + exact kernel, cluster-owner update kernel).  No host
 *            synchronisation inside the loop.
 */
int gsrq_fit_stage(const void *kv, const gsrq_view *view, const float *w, int64_t w_stride_g,
                   const int64_t *fit_tokens, int64_t n_fit, gsrq_codebook *cb, int stage,
                   const float *residual, int iters, uint64_t seed, gsrq_fit_stats *stats,
                   void *workspace, size_t workspace_bytes, gsrq_stream_t stream);

/*
 * Outcome of the last gsrq_fit_stage call that used `workspace` (same view, K, S and fit-subset size as that call; n_fit_tokens:
 * 0 = it fitted on all T tokens).  gsrq_fit_stage(stats = NULL) returns before the GPU has run, so it cannot report what only the
 * kernels find out; this call synchronises `stream` (the fit's stream), reads the per-group error words from the workspace and
 * returns GSRQ_OK, GSRQ_EDEGENERATE (a group had fewer than K distinct non-zero fit rows: its codebook is unspecified) or
 * GSRQ_ECUDA (a CTA of the persistent fit kernel never reached a group barrier within the spin bound; the kernel then stops
 * updating that group's codebook and every CTA of the group leaves the loop).  Each fit clears the words at its start and other
 * gsrq calls may overwrite them, so callers that pass stats == NULL and care call this after each fit, before the next call
 * that is given the same workspace.
 */
int gsrq_fit_status(const void *workspace, const gsrq_view *view, int K, int S, int64_t n_fit_tokens, gsrq_stream_t stream);

/*
 * Encode stages [stage_begin, stage_end) with fixed codebooks (RQ):
 *   for s: a = argmax_k (2 g_k r.s_k - g_k^2) (Eq. 5); code = a; r <- fl32(r - fl32(g_a s_a)).
 * codes       : [S][G][T*M] uint8, stage-major planes (a prefix of stages decodes alone,
 *               PAPER.md:25).  Planes in range are written; when stage_begin > 0 the
 *               planes < stage_begin are READ to rebuild the residual from kv.
 * residual_out: [G][T*M][d] fp32 residual after stage_end-1 (16-byte aligned), or NULL.
 * Kernels     : d == 16, stage_begin == 0, bf16 input with hd/d a power of two (or a dense fp32 tensor):
 *               fused tensor-core passes of up to 4 stages each (the residual stays on the SM within a
 *               pass and is carried in fp32 between passes), each followed by the exact kernel for the
 *               rows it could not decide; otherwise the CUDA-core filter + exact kernel.
 *               Either way every code equals the exact-arithmetic arg-max (ties -> lowest index).
 */
int gsrq_encode(const void *kv, const gsrq_view *view, const gsrq_codebook *cb, int stage_begin,
                int stage_end, uint8_t *codes, float *residual_out, void *workspace,
                size_t workspace_bytes, gsrq_stream_t stream);

/*
 * Decode the first n_stages stages (PAPER.md:56  x ~= sum_l C_l[i_l]; prefix PAPER.md:25):
 *   xhat = ((c0[a0] + c1[a1]) + ...) in fp32, stage order, c_k = fl32(g_k s_k); one
 *   round-to-nearest-even cast to out_view->dtype (reading c-D).
 * kv_out is written through out_view (same striding rules as the input view).
 */
int gsrq_decode(const uint8_t *codes, const gsrq_codebook *cb, int n_stages, void *kv_out,
                const gsrq_view *out_view, gsrq_stream_t stream);

/*
 * Encode-on-append (PAPER.md:443 (i): the "residual quantization ... of newly generated KV vectors" kernel of
 * the paper's decoding loop; K = 256 codes are bytes, so bit-packing is the identity): encode the n_new tokens
 * described by `new_view` (new_view->T = n_new; same G / hd / d / dtype rules as above) with stages [0, n_stages)
 * of cb and store their codes at token positions [t0, t0 + n_new) of the cache's code planes:
 *   codes[(s * G + g) * plane_rows + (t0 + t) * M + m],   plane_rows = T_cache * M   (the layout gsrq_decode reads).
 * One small launch, no workspace; same exact arg-max as gsrq_encode (the codes are identical).
 */
int gsrq_encode_append(const void *kv_new, const gsrq_view *new_view, const gsrq_codebook *cb, int n_stages,
                       uint8_t *codes, int64_t plane_rows, int64_t t0, gsrq_stream_t stream);

/* ---- step-wise entry points (the lock-step parity protocol of DESIGN.md section 6) ---- */

/* One assignment pass over ALL T*M rows of every group against stage `stage` of cb.
 * rows come from `residual` ([G][T*M][d] fp32) when non-NULL, else from kv.
 * mode 0: Eq. 5 score; mode 1: plain projection r.s_k (the init assignment, reading c-I).
 * idx_out: [G][T*M] uint8. */
int gsrq_assign(const void *kv, const gsrq_view *view, const float *residual,
                const gsrq_codebook *cb, int stage, int mode, uint8_t *idx_out, void *workspace,
                size_t workspace_bytes, gsrq_stream_t stream);

/* Test hook: gsrq_assign through the tensor-core filter (d == 16 only) that also dumps the raw
 * filter scores, scores_out [G][T*M][256] fp32 (column k >= K holds -3e38).  Used to validate the
 * filter's error bound E_i against exact arithmetic. */
int gsrq_debug_scores(const void *kv, const gsrq_view *view, const float *residual,
                      const gsrq_codebook *cb, int stage, int mode, float *scores_out,
                      uint8_t *idx_out, void *workspace, size_t workspace_bytes, gsrq_stream_t stream);

/* One update (Eq. 6-8 weighted + safeguards) of stage `stage` of cb from a GIVEN assignment
 * idx [G][T*M] over all rows.  shapes_too = 0 updates gains only (Alg. 1 l.2). */
int gsrq_update(const void *kv, const gsrq_view *view, const float *residual, const float *w,
                int64_t w_stride_g, const uint8_t *idx, gsrq_codebook *cb, int stage,
                int shapes_too, void *workspace, size_t workspace_bytes, gsrq_stream_t stream);

/* The K initial row ids gsrq_fit_stage would draw (local fit-row indices), ids_out [G][K] int64. */
int gsrq_init_ids(const void *kv, const gsrq_view *view, const float *residual,
                  const int64_t *fit_tokens, int64_t n_fit, int K, int stage, uint64_t seed,
                  int64_t *ids_out, void *workspace, size_t workspace_bytes, gsrq_stream_t stream);

/* ---- variants ---- */

/* Log-smoothed gradient weights (PAPER.md:192 Eq. 9; :434 Eq. 10): grad is a tensor laid out like the KV tensor it belongs to
 * (view: dtype, G, T, hd, strides; d is ignored); per head g and token t  w = ||grad[g][t][:]||_2 (stored as fp32),
 * lambda = tau / (median_t w + eps) (median per head; the mean of the two middle values for an even count),
 * w_out[g][t] = log(1 + lambda w).  w_out: device [G][T] fp32 -- pass it to gsrq_fit_stage with w_stride_g = T. */
int gsrq_log_weights(const void *grad, const gsrq_view *view, float tau, float eps, float *w_out, gsrq_stream_t stream);

/* Per-vector gain codes (the alternative reading of "a codeword index plus a gain", reading c-G; BASELINE.json config 0):
 * for each stage s < n_stages:  k = argmax_k r . s_k (lowest index on ties), gamma = fp16(max(0, r . s_k)),
 * r <- fl32(r - fl32(fl32(gamma) s_k)).  Only the shapes of cb are used.  codes [S][G][T*M] uint8 and gains16 [S][G][T*M] IEEE half
 * (as uint16) are written for the stages; residual [G][T*M][d] fp32 is a REQUIRED working buffer and holds the final residual.
 * d in {8, 16, 32}.  workspace as for gsrq_assign (gsrq_workspace_bytes(view, K, S, 0)).  16/d extra bits per element per stage. */
int gsrq_encode_pervector_gain(const void *kv, const gsrq_view *view, const gsrq_codebook *cb, int n_stages, uint8_t *codes,
                               uint16_t *gains16, float *residual, void *workspace, size_t workspace_bytes, gsrq_stream_t stream);

/* xhat = sum_{s < n_stages} fl32(gamma^(s) s^(s)_k), fp32 in stage order, one round-to-nearest-even cast to out_view->dtype. */
int gsrq_decode_pervector_gain(const uint8_t *codes, const uint16_t *gains16, const gsrq_codebook *cb, int n_stages, void *kv_out,
                               const gsrq_view *out_view, gsrq_stream_t stream);

/* Nibble packing for K <= 16 (BASELINE.json config 0 "Codes are 4-bit indices"; "bit-packing"): each of the n_planes
 * rows of N codes becomes ceil(N / 2) bytes, code 2i in the low nibble, code 2i + 1 in the high nibble.  Storage-side only.
 * K is the codebook size the codes were produced with: K > 16 (a code would lose its high bits) returns GSRQ_EINVAL. */
int gsrq_pack_nibbles(const uint8_t *codes, int K, int64_t n_planes, int64_t N, uint8_t *packed, gsrq_stream_t stream);
int gsrq_unpack_nibbles(const uint8_t *packed, int64_t n_planes, int64_t N, uint8_t *codes, gsrq_stream_t stream);

/* Per-subspace codebooks ("an independent codebook per subspace"): no separate entry point -- subspace m of a
 * [G][T][hd] tensor is the view {G, T, hd' = d, d, stride_g, stride_t} on the pointer kv + m * d elements, and a head-inner
 * [T][G][hd] tensor is ONE view with G' = G * M groups, hd' = d, stride_g' = d (tests/test_gpu_variants.py). */

/* ---- decode fused into attention (PAPER.md:443 (ii), :445) ---- */

/* Scratch of gsrq_attention_decode for B sequences of at most max_len tokens (host function, no CUDA calls). */
size_t gsrq_attention_workspace_bytes(int B, int Hq, int G, int64_t max_len);

/*
 * One decoding step of grouped-query attention computed straight from the GSRQ codes of the K and V cache, without writing the
 * dequantised cache (PAPER.md:443 (ii): "bit-unpacking, dequantization, RoPE, and attention computation ... without materializing
 * intermediate FP16 tensors"): for sequence b and query head h (KV head g = h / (Hq / G)), over the tokens t of the sequence,
 *     out[b][h] = sum_t softmax_t(scale * q[b][h] . k_t) * vhat_t,
 *     khat_t = sum_{s < k_stages} cK^(s)[codes], vhat_t = sum_{s < v_stages} cV^(s)[codes]  (fp32, stage order, as gsrq_decode; no cast),
 *     k_t = khat_t (rope_theta == 0: keys were quantised after the rotary embedding) or RoPE(khat_t, t) (rope_theta > 0: rotate-half
 *     convention, angle = t * rope_theta^(-2 i / hd), t counted from the sequence's first token; q is given already rotated).
 * q        : [B][Hq][hd] fp32.            out: [B][Hq][hd] fp32 (zeros for an empty sequence).
 * k_codes / v_codes: the cache's code planes as gsrq_encode / gsrq_encode_append write them, [S][G][plane_rows], row = token * M + m
 *            (8-byte aligned); k_cb / v_cb their codebooks; k_stages / v_stages: prefix of stages used.
 * seq_start, seq_len: device [B] int64: first token and number of tokens of each sequence inside the planes; max_len >= every seq_len
 *            (host value, sizes the split of the token range over CTAs).  A sequence with a negative start or length, or one that
 *            reaches beyond plane_rows / 8 tokens, is not read: it is served as an empty sequence (zeros).
 * B, G <= 65535; the codebooks' shapes arrays must be 16-byte aligned (GSRQ_EINVAL otherwise).  Code bytes >= K select a zero
 *            codeword here; the stand-alone decodes clamp them to K - 1 (cold paths) -- either way nothing outside the codebook is read.
 * This build serves hd = 128, K <= 256, Hq / G <= 8, with d = 16 and 1..4 stages (table-lookup kernels, shared-memory codeword tables)
 * or d = 128 and 1..32 stages (the paper's operating point: D = 128, R = 12 / 16 / 32; row = token, plane_rows =
 * tokens in the planes; a dequantising kernel that reads the codeword rows from L2 -- functional, far from the d = 16 kernels'
 * speed).  q must be 16-byte aligned.  fp32 arithmetic, no atomics: bit-reproducible.
 */
int gsrq_attention_decode(const float *q, const uint8_t *k_codes, const gsrq_codebook *k_cb, int k_stages, const uint8_t *v_codes,
                          const gsrq_codebook *v_cb, int v_stages, int64_t plane_rows, const int64_t *seq_start, const int64_t *seq_len,
                          int64_t max_len, int B, int Hq, int G, int hd, int d, float scale, float rope_theta, float *out,
                          void *workspace, size_t workspace_bytes, gsrq_stream_t stream);

/*
 * gsrq_attention_decode for callers that cannot provide scratch memory.
 *
 * Who this is for: code that runs where device memory can no longer be obtained, so that it has no workspace to pass to
 * gsrq_attention_decode -- a serving loop whose memory manager has claimed the whole GPU for the KV cache and hands nothing back;
 * a plug-in called from inside somebody else's stream capture or latency-critical section, where cudaMalloc / cudaFree are not
 * permitted (they synchronise the device, and are not allowed while a stream is capturing); a host that forbids allocation after
 * start-up.  This call, and everything under it, calls no cudaMalloc, no cudaFree, no memory pool and no other allocating routine:
 * the per-split partial results go to a fixed buffer of GSRQ_ATTENTION_STATIC_SCRATCH_BYTES that is part of the library image.
 * Every GPU on which the library's kernels are loaded holds that buffer from then until the process exits, used or not.
 *
 * Arguments, arithmetic and results are those of gsrq_attention_decode (bit-identical: same kernels, same split of the token range),
 * without `workspace` / `workspace_bytes`; it serves the d = 16 shapes (1..4 stages) only.  The caller still owns and passes q, the code planes, the codebooks,
 * seq_start / seq_len and out (device pointers).
 *
 * Limit: B * G * n_split * (Hq / G) * 130 * 4 bytes must fit in the buffer, n_split being the library's split of the token range
 * (at most 4 * SM count / (B * G), at most one per 2048 tokens of max_len, at least 1).  With LLaMA-3-8B's 8 KV heads and 4 query
 * heads per KV head that is every batch up to 252 sequences (batch 8 x 131072 tokens needs 1.2 MiB).  A larger request returns
 * GSRQ_EWORKSPACE with the needed and available sizes in gsrq_last_error(), and launches nothing; use gsrq_attention_decode then.
 *
 * First call on each device: looks up the buffer's device address (cudaGetSymbolAddress, with the caller's current device), which
 * can make the CUDA runtime load the library's device code.  Make this first call at start-up on every device that will be used,
 * outside any stream capture; later calls only read the cached address.
 *
 * One buffer per device, shared by every call in the process, and not cleared between calls (no entry has to start at zero:
 * each call overwrites every entry it later reads).  Two calls that can run at the same time on one GPU -- issued to different
 * streams without an ordering between them, or from two threads -- overwrite each other's partial results and return garbage:
 * order them (same stream, or an event).  Calls on different GPUs are independent.  The launches of this entry point are counted by
 * gsrq_launch_count() but are never event-timed by gsrq_profile_enable().
 */
#define GSRQ_ATTENTION_STATIC_SCRATCH_BYTES (4u << 20)
size_t gsrq_attention_static_scratch_bytes(void); /* == GSRQ_ATTENTION_STATIC_SCRATCH_BYTES; host function, no CUDA calls */
int gsrq_attention_decode_static(const float *q, const uint8_t *k_codes, const gsrq_codebook *k_cb, int k_stages, const uint8_t *v_codes,
                                 const gsrq_codebook *v_cb, int v_stages, int64_t plane_rows, const int64_t *seq_start,
                                 const int64_t *seq_len, int64_t max_len, int B, int Hq, int G, int hd, int d, float scale,
                                 float rope_theta, float *out, gsrq_stream_t stream);

/* ---- stand-alone clustering of fp32 rows: GSKM against the K-means baseline (section 6.1, :200-212; section 4, :60-85) ---- */

/* Scratch for the three calls below (host function, no CUDA calls); 0 on bad arguments. */
size_t gsrq_cluster_workspace_bytes(int64_t N, int d, int K);

/*
 * Learn a codebook of K prototypes on x [N][d] fp32 (device, 16-byte aligned; d a multiple of 4, d <= 256; K <= 4096), one group:
 *   method 0: weighted GSKM, Algorithm 1 exactly as gsrq_fit_stage runs it (seeded init, Eq. 5 / 7 / 8, safeguards, early exit);
 *   method 1: standard weighted K-means "KM" (l2 assignment, arithmetic-mean centroid; Lloyd iterations from the
 *             same K seeded rows; ties -> lowest index; an empty cluster keeps its centroid).
 * w: [N] fp32 per-row weights or NULL.  Out: shapes [K][d], gains [K] (KM: shapes holds the centroids mu_k, gains = 1), idx_out [N]
 * uint16 = the assignment of the last iteration run, stats (host, one struct, or NULL; when given the call synchronises).
 * Every assignment is the exact arg-max / arg-min (fp64, the definition's operation order); sums in fp64, fixed order.
 */
int gsrq_cluster_fit(const float *x, const float *w, int64_t N, int d, int K, int iters, uint64_t seed, int method, float *shapes,
                     float *gains, uint16_t *idx_out, gsrq_fit_stats *stats, void *workspace, size_t workspace_bytes,
                     gsrq_stream_t stream);

/* One assignment of every row against a given codebook (method as above): idx_out [N] uint16. */
int gsrq_cluster_assign(const float *x, int64_t N, int d, int K, int method, const float *shapes, const float *gains,
                        uint16_t *idx_out, gsrq_stream_t stream);

/* Quality of the reconstruction xhat_i = prototype of idx_i (KM: mu_k; GSKM: fl32(g_k s_k)), PAPER.md:202 and :85:
 * out_host[0] = MSE = E||x - xhat||^2, [1] = gain error E| ||x|| - ||xhat|| |, [2] = cosine similarity E cos(x, xhat),
 * [3] = shrinkage ratio E||xhat||^2 / E||x||^2.  out_host is a HOST array of 4 doubles; the call synchronises. */
int gsrq_cluster_metrics(const float *x, int64_t N, int d, int K, int method, const float *shapes, const float *gains,
                         const uint16_t *idx, double *out_host, void *workspace, size_t workspace_bytes, gsrq_stream_t stream);

/* ---- host-buffer convenience (end-to-end measurement: H2D + kernels + D2H inside) ---- */

/* gsrq_encode on HOST buffers: kv_host and codes_host are host pointers (pinned or pageable);
 * cb holds DEVICE codebooks.  Allocates device scratch for the duration of the call, copies
 * kv in, encodes [0,S), copies all S code planes out, synchronises. */
int gsrq_encode_host(const void *kv_host, const gsrq_view *view, const gsrq_codebook *cb,
                     uint8_t *codes_host);

/* gsrq_decode on HOST buffers: codes_host in, kv_out_host out (contiguous per out_view). */
int gsrq_decode_host(const uint8_t *codes_host, const gsrq_codebook *cb, int n_stages,
                     void *kv_out_host, const gsrq_view *out_view);

/* The whole hot path on HOST buffers, as one call (the end-to-end measurement): copies kv_host
 * (dense, laid out as `view` says), w_host ([T] or NULL) and fit_tokens_host ([G][n_fit] sorted token ids,
 * or NULL = fit on all T tokens) to the device.  Fit on all tokens: for each stage s < S gsrq_fit_stage
 * (`iters`, `seed`) + gsrq_encode of that stage (its residual feeds the next fit).  Fit on a token subset:
 * the S fits (each re-deriving its residual on the fit rows), then one fused gsrq_encode of all stages.  Then,
 * when kv_out_host != NULL, gsrq_decode of all S stages; copies shapes [G][S][K][d], gains [G][S][K],
 * codes [S][G][T*M] (and the decoded tensor) back to the host and synchronises.  Returns GSRQ_EDEGENERATE if a
 * group could not be initialised (fewer than K distinct non-zero fit rows).  Device memory comes from the
 * library's private pool (see the conventions at the top). */
int gsrq_pipeline_host(const void *kv_host, const gsrq_view *view, const float *w_host, const int64_t *fit_tokens_host,
                       int64_t n_fit, int K, int S, int iters, uint64_t seed, float *shapes_host, float *gains_host,
                       uint8_t *codes_host, void *kv_out_host);

/* gsrq_pipeline_host for n tensors of the same view (a layer's K and V cache, several layers, ...), pipelined: the tensors
 * alternate between two streams, so that tensor i + 1 is uploaded while tensor i is fitted, encoded, decoded and downloaded (both
 * copy directions and the SMs busy at once; uploads follow one another, each at full link speed).  Every array has n entries:
 * kv_host[i], shapes_host[i], gains_host[i], codes_host[i] as in gsrq_pipeline_host; w_host, fit_tokens_host, kv_out_host may be
 * NULL or hold NULL entries (no weights / fit on all tokens / no decode); n_fit, K, S, iters, seed are shared.  The host
 * buffers should be pinned: a copy from or to pageable memory blocks the calling thread and serialises the tensors.  Results
 * are identical to n calls of gsrq_pipeline_host.  Returns the first tensor's error, if any; synchronises. */
int gsrq_pipeline_host_batch(int n, const void *const *kv_host, const gsrq_view *view, const float *const *w_host,
                             const int64_t *const *fit_tokens_host, int64_t n_fit, int K, int S, int iters, uint64_t seed,
                             float *const *shapes_host, float *const *gains_host, uint8_t *const *codes_host, void *const *kv_out_host);

/* Free the device memory the *_host entry points keep between calls (current device). */
void gsrq_release_host_pool(void);

/* ---- measurement hooks (host functions) ---- */

#define GSRQ_N_KERNEL_CLASSES 7 /* 0 prep, 1 score (fit assignment passes; CUDA-core encode), 2 refine (exact path kernel), 3 update, 4 misc, 5 decode, 6 encode (fused tensor-core encode) */

/* When on, every kernel launch of this library is bracketed by a CUDA event pair on its stream. */
void gsrq_profile_enable(int on);
/* Synchronise the recorded events; per kernel class return summed device ms and launch counts
 * since the last read (arrays of GSRQ_N_KERNEL_CLASSES, either may be NULL); clears the record. */
int gsrq_profile_read(double *ms_by_class, int64_t *launches_by_class);
/* Kernels launched by this library in this process so far. */
int64_t gsrq_launch_count(void);

/* Thread-local message of the last error returned on this thread ("" if none). */
const char *gsrq_last_error(void);

/* Library version string, e.g. "gsrq-b200 0.1 (sm_100a)". */
const char *gsrq_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GSRQ_H_ */
