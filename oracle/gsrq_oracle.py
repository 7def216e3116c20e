"""ctypes wrapper around oracle/gsrq_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / ``--impl reference``
legs may import this module.  It imports nothing from paper_2607_01065_b200 (the
CUDA path) and the CUDA path imports nothing from here.

The C file holds all of the method's arithmetic (one codebook group, one stage per
call); this wrapper only marshals numpy arrays and loops over groups and stages in
the order the paper gives:  PQ split into sub-vectors of dim d,
then for each residual stage: fit a codebook with weighted GSKM on the fit rows
(Alg. 1), encode every row, subtract.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gsrq_oracle.c"
_SRC_KM = _HERE / "km_oracle.c"      # K-means baseline + quality metrics (section 6.1)
_SO = _HERE / "build" / "libgsrq_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (no fast-math, no FMA contraction)."""
    if force or not _SO.exists() or _SO.stat().st_mtime < max(_SRC.stat().st_mtime, _SRC_KM.stat().st_mtime):
        _SO.parent.mkdir(exist_ok=True)
        tmp = _SO.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-fno-fast-math", "-o", str(tmp), str(_SRC), str(_SRC_KM), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.gsrq_oracle_wdist.restype = C.c_double
        _lib.km_oracle_wdist.restype = C.c_double
        _lib.gsrq_oracle_splitmix64_next.restype = C.c_uint64
    return _lib


def n_threads() -> int:
    """Threads the assignment step uses (OpenMP default = visible cores unless OMP_NUM_THREADS)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else len(os.sched_getaffinity(0))


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def splitmix64(seed: int, n: int):
    st = C.c_uint64(seed)
    return [int(lib().gsrq_oracle_splitmix64_next(C.byref(st))) for _ in range(n)]


def init_ids(r, K, seed, group=0, G=1, stage=0):
    r = _f32(r)
    ids = np.zeros(K, dtype=np.int64)
    rc = lib().gsrq_oracle_init_ids(_p(r, C.c_float), C.c_int64(r.shape[0]), r.shape[1], K,
                                    C.c_uint64(seed), group, G, stage, _p(ids, C.c_int64))
    if rc != 0:
        raise ValueError("degenerate input: fewer than K distinct non-zero rows")
    return ids


def assign(r, s, g=None):
    """Eq. 5 assignment (g given) or max projection (g None). Returns idx, best, second."""
    r, s = _f32(r), _f32(s)
    g = _f32(g) if g is not None else None
    N, d = r.shape
    K = s.shape[0]
    idx = np.zeros(N, dtype=np.int32)
    best = np.zeros(N, dtype=np.float64)
    second = np.zeros(N, dtype=np.float64)
    lib().gsrq_oracle_assign(_p(r, C.c_float), C.c_int64(N), d, _p(s, C.c_float), _p(g, C.c_float), K,
                             _p(idx, C.c_int32), _p(best, C.c_double), _p(second, C.c_double))
    return idx, best, second


def update(r, w, idx, s, g, shapes_too=True):
    """Eq. 6-8 update given an assignment. Returns new (s, g, n_empty, cnt)."""
    r = _f32(r)
    w = _f32(w) if w is not None else None
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    s, g = _f32(s).copy(), _f32(g).copy()
    N, d = r.shape
    K = s.shape[0]
    cnt = np.zeros(K, dtype=np.int64)
    ne = lib().gsrq_oracle_update(_p(r, C.c_float), _p(w, C.c_float), C.c_int64(N), d, _p(idx, C.c_int32),
                                  K, _p(s, C.c_float), _p(g, C.c_float), int(bool(shapes_too)),
                                  _p(cnt, C.c_int64))
    return s, g, int(ne), cnt


def wdist(r, w, idx, s, g) -> float:
    r, s, g = _f32(r), _f32(s), _f32(g)
    w = _f32(w) if w is not None else None
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    return float(lib().gsrq_oracle_wdist(_p(r, C.c_float), _p(w, C.c_float), C.c_int64(r.shape[0]),
                                         r.shape[1], _p(idx, C.c_int32), _p(s, C.c_float), _p(g, C.c_float)))


def fit_stage(r, w, K, iters, seed, group=0, G=1, stage=0):
    """Algorithm 1 on one group's rows. Returns a dict."""
    r = _f32(r)
    w = _f32(w) if w is not None else None
    N, d = r.shape
    s = np.zeros((K, d), dtype=np.float32)
    g = np.zeros(K, dtype=np.float32)
    idx = np.zeros(N, dtype=np.int32)
    J = np.full(max(iters, 1), np.nan, dtype=np.float64)
    ch = np.full(max(iters, 1), -1, dtype=np.int64)
    it = C.c_int32(0)
    ne = C.c_int32(0)
    ids = np.zeros(K, dtype=np.int64)
    rc = lib().gsrq_oracle_fit_stage(_p(r, C.c_float), _p(w, C.c_float), C.c_int64(N), d, K, iters,
                                     C.c_uint64(seed), group, G, stage, _p(s, C.c_float), _p(g, C.c_float),
                                     _p(idx, C.c_int32), _p(J, C.c_double), _p(ch, C.c_int64),
                                     C.byref(it), C.byref(ne), _p(ids, C.c_int64))
    if rc != 0:
        raise ValueError("degenerate input: fewer than K distinct non-zero rows")
    return dict(shapes=s, gains=g, idx_last=idx, J_assign=J[:it.value], changed=ch[:it.value],
                iters_run=it.value, n_empty_last=ne.value, init_ids=ids)


def encode_stage(r, s, g):
    """One RQ stage on rows r (not modified). Returns codes, new residual, best, second."""
    r = _f32(r).copy()
    s, g = _f32(s), _f32(g)
    N, d = r.shape
    codes = np.zeros(N, dtype=np.uint8)
    best = np.zeros(N, dtype=np.float64)
    second = np.zeros(N, dtype=np.float64)
    lib().gsrq_oracle_encode_stage(_p(r, C.c_float), C.c_int64(N), d, _p(s, C.c_float), _p(g, C.c_float),
                                   s.shape[0], _p(codes, C.c_uint8), _p(best, C.c_double), _p(second, C.c_double))
    return codes, r, best, second


def decode_rows(codes, s, g, S_used=None):
    """codes [S][N] uint8, s [S][K][d], g [S][K] -> fp32 [N][d], stage-order fp32 sum."""
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    s, g = _f32(s), _f32(g)
    S, N = codes.shape
    K, d = s.shape[1], s.shape[2]
    S_used = S if S_used is None else S_used
    out = np.zeros((N, d), dtype=np.float32)
    lib().gsrq_oracle_decode(_p(codes, C.c_uint8), C.c_int64(N), d, _p(s, C.c_float), _p(g, C.c_float),
                             K, S_used, _p(out, C.c_float))
    return out


def f32_to_bf16_bits(x):
    x = _f32(x)
    out = np.zeros(x.shape, dtype=np.uint16)
    lib().gsrq_oracle_f32_to_bf16(_p(x, C.c_float), C.c_int64(x.size), _p(out, C.c_uint16))
    return out


def bf16_bits_to_f32(b):
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)


# ---------------------------------------------------------------------------
# Whole-tensor drivers (layout only; no arithmetic of the method lives here)
# ---------------------------------------------------------------------------
def rows_of(x, d):
    """PQ split: x [G][T][hd] -> rows [G][T*M][d], M = hd/d, row = t*M + m."""
    G, T, hd = x.shape
    assert hd % d == 0
    return _f32(x).reshape(G, T * (hd // d), d)


def gsrq_fit_encode(x, w_tok, d, K, S, iters, seed=0, fit_tokens=None, encode=True):
    """Full GSRQ encoder on x [G][T][hd] (fp32 values; bf16 inputs are passed as their exact fp32).

    w_tok: [T] or [G][T] per-token weights (a sub-vector inherits its token's weight) or None.
    fit_tokens: [G][n_fit] sorted token ids (codebooks are fitted on those tokens' rows), None = all.
    Returns shapes [G][S][K][d], gains [G][S][K], codes [S][G][T*M], residual [G][T*M][d],
    and per (group, stage) stats.
    """
    G, T, hd = x.shape
    M = hd // d
    rows = rows_of(x, d).copy()
    Ng = T * M
    shapes = np.zeros((G, S, K, d), dtype=np.float32)
    gains = np.zeros((G, S, K), dtype=np.float32)
    codes = np.zeros((S, G, Ng), dtype=np.uint8)
    best = np.zeros((S, G, Ng), dtype=np.float64)
    second = np.zeros((S, G, Ng), dtype=np.float64)
    stats = [[None] * S for _ in range(G)]
    for g_ in range(G):
        if w_tok is None:
            w_t = np.ones(T, dtype=np.float32)
        else:
            w_t = _f32(w_tok if np.ndim(w_tok) == 1 else w_tok[g_])
        if fit_tokens is None:
            fit_rows = None
            w_fit = np.repeat(w_t, M)
        else:
            ft = np.asarray(fit_tokens[g_], dtype=np.int64)
            fit_rows = (ft[:, None] * M + np.arange(M)[None, :]).reshape(-1)
            w_fit = np.repeat(w_t[ft], M)
        for st in range(S):
            r_fit = rows[g_] if fit_rows is None else rows[g_][fit_rows]
            f = fit_stage(r_fit, w_fit, K, iters, seed, group=g_, G=G, stage=st)
            shapes[g_, st], gains[g_, st] = f["shapes"], f["gains"]
            stats[g_][st] = f
            if encode or st + 1 < S:
                codes[st, g_], rows[g_], best[st, g_], second[st, g_] = encode_stage(rows[g_], f["shapes"], f["gains"])
    return dict(shapes=shapes, gains=gains, codes=codes, residual=rows, best=best, second=second, stats=stats)


def encode(x, shapes, gains, d, stage_begin=0, stage_end=None, residual_in=None):
    """Encode with fixed codebooks. Returns codes [S'][G][Ng], residual, best, second."""
    G, T, hd = x.shape
    S = shapes.shape[1]
    stage_end = S if stage_end is None else stage_end
    rows = rows_of(x, d).copy() if residual_in is None else _f32(residual_in).copy()
    Ng = rows.shape[1]
    n = stage_end - stage_begin
    codes = np.zeros((n, G, Ng), dtype=np.uint8)
    best = np.zeros((n, G, Ng), dtype=np.float64)
    second = np.zeros((n, G, Ng), dtype=np.float64)
    for g_ in range(G):
        for q, st in enumerate(range(stage_begin, stage_end)):
            codes[q, g_], rows[g_], best[q, g_], second[q, g_] = encode_stage(rows[g_], shapes[g_, st], gains[g_, st])
    return codes, rows, best, second


def decode(codes, shapes, gains, hd, S_used=None, bf16=True):
    """codes [S][G][Ng] -> x_hat [G][T][hd]; fp32 sum in stage order, then one RN-even cast (c-D).

    Returns fp32 values (bf16-exact when bf16=True) and, when bf16, the uint16 bit patterns.
    """
    S, G, Ng = codes.shape
    d = shapes.shape[3]
    M = hd // d
    T = Ng // M
    out = np.zeros((G, Ng, d), dtype=np.float32)
    for g_ in range(G):
        out[g_] = decode_rows(codes[:, g_], shapes[g_], gains[g_], S_used)
    out = out.reshape(G, T, hd)
    if not bf16:
        return out, None
    bits = f32_to_bf16_bits(out)
    return bf16_bits_to_f32(bits), bits


# ---- K-means baseline and quality metrics (oracle/km_oracle.c; section 6.1, :200-212) ----
def km_assign(x, mu):
    """argmin_k ||x_i - mu_k||^2, lowest k on ties. Returns idx, squared distance."""
    x, mu = _f32(x), _f32(mu)
    N, d = x.shape
    idx = np.zeros(N, dtype=np.int32)
    best = np.zeros(N, dtype=np.float64)
    lib().km_oracle_assign(_p(x, C.c_float), C.c_int64(N), d, _p(mu, C.c_float), mu.shape[0], _p(idx, C.c_int32), _p(best, C.c_double))
    return idx, best


def km_update(x, w, idx, mu):
    """mu_k = weighted mean of the cluster (empty cluster keeps mu_k). Returns new mu, n_empty."""
    x, mu = _f32(x), _f32(mu).copy()
    w = _f32(w) if w is not None else None
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    ne = lib().km_oracle_update(_p(x, C.c_float), _p(w, C.c_float), C.c_int64(x.shape[0]), x.shape[1], _p(idx, C.c_int32), mu.shape[0], _p(mu, C.c_float))
    return mu, int(ne)


def km_fit(x, w, K, iters, seed):
    """Lloyd K-means from K seeded distinct rows. Returns a dict."""
    x = _f32(x)
    w = _f32(w) if w is not None else None
    N, d = x.shape
    mu = np.zeros((K, d), dtype=np.float32)
    idx = np.zeros(N, dtype=np.int32)
    J = np.full(max(iters, 1), np.nan, dtype=np.float64)
    ch = np.full(max(iters, 1), -1, dtype=np.int64)
    it, ne = C.c_int32(0), C.c_int32(0)
    rc = lib().km_oracle_fit(_p(x, C.c_float), _p(w, C.c_float), C.c_int64(N), d, K, iters, C.c_uint64(seed), _p(mu, C.c_float),
                             _p(idx, C.c_int32), _p(J, C.c_double), _p(ch, C.c_int64), C.byref(it), C.byref(ne))
    if rc != 0:
        raise ValueError("degenerate input: fewer than K distinct non-zero rows")
    return dict(mu=mu, idx_last=idx, J_assign=J[:it.value], changed=ch[:it.value], iters_run=it.value, n_empty_last=ne.value)


def metrics(x, proto, idx):
    """MSE, gain error, cosine similarity, shrinkage ratio of the reconstruction xhat_i = proto[idx_i]."""
    x, proto = _f32(x), _f32(proto)
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    out = np.zeros(4, dtype=np.float64)
    lib().km_oracle_metrics(_p(x, C.c_float), C.c_int64(x.shape[0]), x.shape[1], _p(proto, C.c_float), _p(idx, C.c_int32), _p(out, C.c_double))
    return dict(mse=float(out[0]), gain_err=float(out[1]), cosine=float(out[2]), shrinkage=float(out[3]))
