"""Thin ctypes binding over libgsrq (include/gsrq.h): argument marshalling only.

Functions carry the C names.  Tensors are torch CUDA tensors used purely as device
memory; the current torch CUDA stream is passed as the stream.  There is no fallback:
if the library is not built, or a call fails, this raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import torch

from . import build as _build

GSRQ_MAX_ITERS = 128
GSRQ_F32, GSRQ_BF16 = 0, 1
_STATUS = {0: "GSRQ_OK", -1: "GSRQ_EINVAL", -2: "GSRQ_EUNSUPPORTED", -3: "GSRQ_EWORKSPACE",
           -4: "GSRQ_ECUDA", -5: "GSRQ_EDEGENERATE"}


class GsrqError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_STATUS.get(code, code)}: {msg}")
        self.code = code


class gsrq_view(C.Structure):
    _fields_ = [("dtype", C.c_int32), ("G", C.c_int32), ("T", C.c_int64), ("hd", C.c_int32), ("d", C.c_int32),
                ("stride_g", C.c_int64), ("stride_t", C.c_int64)]


class gsrq_codebook(C.Structure):
    _fields_ = [("K", C.c_int32), ("S", C.c_int32), ("shapes", C.c_void_p), ("gains", C.c_void_p)]


class gsrq_fit_stats(C.Structure):
    _fields_ = [("iters_run", C.c_int32), ("n_empty_last", C.c_int32), ("n_changed_last", C.c_int64),
                ("n_refined", C.c_int64), ("wdist_after_assign", C.c_double * GSRQ_MAX_ITERS),
                ("n_changed", C.c_int64 * GSRQ_MAX_ITERS)]


_lib = None
EXPORTS = ["gsrq_log_weights", "gsrq_encode_pervector_gain", "gsrq_decode_pervector_gain", "gsrq_pack_nibbles", "gsrq_unpack_nibbles",
           "gsrq_attention_workspace_bytes", "gsrq_attention_decode", "gsrq_attention_static_scratch_bytes", "gsrq_attention_decode_static", "gsrq_cluster_workspace_bytes", "gsrq_cluster_fit", "gsrq_cluster_assign", "gsrq_cluster_metrics", "gsrq_workspace_bytes", "gsrq_fit_stage", "gsrq_fit_status", "gsrq_encode", "gsrq_decode", "gsrq_encode_append", "gsrq_assign", "gsrq_update",
           "gsrq_init_ids", "gsrq_debug_scores", "gsrq_encode_host", "gsrq_decode_host", "gsrq_pipeline_host", "gsrq_pipeline_host_batch", "gsrq_release_host_pool", "gsrq_profile_enable",
           "gsrq_profile_read", "gsrq_launch_count", "gsrq_last_error", "gsrq_version"]


def lib_path() -> Path:
    return _build.LIB


def lib():
    """Load libgsrq.so (built in-tree by paper_2607_01065_b200.build). Fails loudly if absent."""
    global _lib
    if _lib is None:
        p = lib_path()
        if not p.exists():
            raise ImportError(f"{p} is not built: run `python -c 'import __graft_entry__ as g; g.build()'`")
        _lib = C.CDLL(str(p))
        _lib.gsrq_workspace_bytes.restype = C.c_size_t
        _lib.gsrq_cluster_workspace_bytes.restype = C.c_size_t
        _lib.gsrq_attention_workspace_bytes.restype = C.c_size_t
        _lib.gsrq_attention_static_scratch_bytes.restype = C.c_size_t
        _lib.gsrq_last_error.restype = C.c_char_p
        _lib.gsrq_version.restype = C.c_char_p
        _lib.gsrq_launch_count.restype = C.c_int64
    return _lib


def _check(rc):
    if rc != 0:
        raise GsrqError(rc, lib().gsrq_last_error().decode())


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def view_of(x: torch.Tensor, d: int, head_inner: bool = False) -> gsrq_view:
    """View for a [G][T][hd] tensor (or [T][G][hd] when head_inner)."""
    dt = {torch.float32: GSRQ_F32, torch.bfloat16: GSRQ_BF16}[x.dtype]
    if head_inner:
        T, G, hd = x.shape
        sg, st = x.stride(1), x.stride(0)
    else:
        G, T, hd = x.shape
        sg, st = x.stride(0), x.stride(1)
    assert x.stride(2) == 1
    return gsrq_view(dt, G, T, hd, d, sg, st)


def codebook_of(shapes: torch.Tensor, gains: torch.Tensor) -> gsrq_codebook:
    """shapes [G][S][K][d] fp32, gains [G][S][K] fp32, contiguous CUDA tensors."""
    assert shapes.is_contiguous() and gains.is_contiguous() and shapes.dtype == torch.float32
    return gsrq_codebook(shapes.shape[2], shapes.shape[1], shapes.data_ptr(), gains.data_ptr())


def gsrq_version() -> str:
    return lib().gsrq_version().decode()


def gsrq_workspace_bytes(view: gsrq_view, K: int, S: int, n_fit_tokens: int = 0) -> int:
    n = lib().gsrq_workspace_bytes(C.byref(view), K, S, C.c_int64(n_fit_tokens))
    if n == 0:
        raise GsrqError(-1, lib().gsrq_last_error().decode())
    return n


def workspace(view: gsrq_view, K: int, S: int, n_fit_tokens: int = 0, device="cuda") -> torch.Tensor:
    return torch.empty(gsrq_workspace_bytes(view, K, S, n_fit_tokens), dtype=torch.uint8, device=device)


def gsrq_fit_stage(kv, view, w, w_stride_g, fit_tokens, cb, stage, residual, iters, seed, ws, want_stats=True):
    G = view.G
    stats = (gsrq_fit_stats * G)() if want_stats else None
    n_fit = 0 if fit_tokens is None else fit_tokens.shape[1]
    rc = lib().gsrq_fit_stage(_ptr(kv), C.byref(view), _ptr(w), C.c_int64(w_stride_g), _ptr(fit_tokens),
                              C.c_int64(n_fit), C.byref(cb), stage, _ptr(residual), iters, C.c_uint64(seed),
                              stats, _ptr(ws), C.c_size_t(ws.numel()), _stream())
    _check(rc)
    return stats


def gsrq_fit_status(ws, view, K, S, n_fit_tokens=0):
    """Raise GsrqError if the last gsrq_fit_stage on this workspace hit a degenerate group or a barrier timeout (synchronises)."""
    _check(lib().gsrq_fit_status(_ptr(ws), C.byref(view), K, S, C.c_int64(n_fit_tokens), _stream()))


def gsrq_encode(kv, view, cb, stage_begin, stage_end, codes, residual_out, ws):
    _check(lib().gsrq_encode(_ptr(kv), C.byref(view), C.byref(cb), stage_begin, stage_end, _ptr(codes),
                             _ptr(residual_out), _ptr(ws), C.c_size_t(ws.numel()), _stream()))


def gsrq_encode_append(kv_new, new_view, cb, n_stages, codes, plane_rows, t0):
    _check(lib().gsrq_encode_append(_ptr(kv_new), C.byref(new_view), C.byref(cb), n_stages, _ptr(codes),
                                    C.c_int64(plane_rows), C.c_int64(t0), _stream()))


def gsrq_decode(codes, cb, n_stages, kv_out, out_view):
    _check(lib().gsrq_decode(_ptr(codes), C.byref(cb), n_stages, _ptr(kv_out), C.byref(out_view), _stream()))


def gsrq_assign(kv, view, residual, cb, stage, mode, idx_out, ws):
    _check(lib().gsrq_assign(_ptr(kv), C.byref(view), _ptr(residual), C.byref(cb), stage, mode, _ptr(idx_out),
                             _ptr(ws), C.c_size_t(ws.numel()), _stream()))


def gsrq_debug_scores(kv, view, residual, cb, stage, mode, scores_out, idx_out, ws):
    _check(lib().gsrq_debug_scores(_ptr(kv), C.byref(view), _ptr(residual), C.byref(cb), stage, mode, _ptr(scores_out),
                                   _ptr(idx_out), _ptr(ws), C.c_size_t(ws.numel()), _stream()))


def gsrq_update(kv, view, residual, w, w_stride_g, idx, cb, stage, shapes_too, ws):
    _check(lib().gsrq_update(_ptr(kv), C.byref(view), _ptr(residual), _ptr(w), C.c_int64(w_stride_g), _ptr(idx),
                             C.byref(cb), stage, int(shapes_too), _ptr(ws), C.c_size_t(ws.numel()), _stream()))


def gsrq_init_ids(kv, view, residual, fit_tokens, K, stage, seed, ids_out, ws):
    n_fit = 0 if fit_tokens is None else fit_tokens.shape[1]
    _check(lib().gsrq_init_ids(_ptr(kv), C.byref(view), _ptr(residual), _ptr(fit_tokens), C.c_int64(n_fit), K, stage,
                               C.c_uint64(seed), _ptr(ids_out), _ptr(ws), C.c_size_t(ws.numel()), _stream()))


def gsrq_attention_decode(q, k_codes, k_cb, k_stages, v_codes, v_cb, v_stages, plane_rows, seq_start, seq_len, max_len, G, d, scale,
                          rope_theta, out, ws=None):
    """q [B][Hq][hd] fp32, codes [S][G][plane_rows] uint8, seq_start / seq_len int64 [B] CUDA tensors; out [B][Hq][hd] fp32."""
    Bq, Hq, hd = q.shape
    if ws is None:
        n = lib().gsrq_attention_workspace_bytes(Bq, Hq, G, C.c_int64(max_len))
        if n == 0:
            raise GsrqError(-1, lib().gsrq_last_error().decode())
        ws = torch.empty(n, dtype=torch.uint8, device="cuda")
    _check(lib().gsrq_attention_decode(_ptr(q), _ptr(k_codes), C.byref(k_cb), k_stages, _ptr(v_codes), C.byref(v_cb), v_stages,
                                       C.c_int64(plane_rows), _ptr(seq_start), _ptr(seq_len), C.c_int64(max_len), Bq, Hq, G, hd, d,
                                       C.c_float(scale), C.c_float(rope_theta), _ptr(out), _ptr(ws), C.c_size_t(ws.numel()), _stream()))
    return ws


def gsrq_attention_static_scratch_bytes():
    return int(lib().gsrq_attention_static_scratch_bytes())


def gsrq_attention_decode_static(q, k_codes, k_cb, k_stages, v_codes, v_cb, v_stages, plane_rows, seq_start, seq_len, max_len, G, d, scale,
                                 rope_theta, out):
    """gsrq_attention_decode without a workspace: for callers that cannot obtain device memory (an engine that has given the whole
    GPU to its KV cache, code running inside a stream capture, a no-allocation-after-start-up host).  The partial results go to a
    fixed 4 MiB buffer inside the library; larger requests raise GSRQ_EWORKSPACE.  Same tensors and results as gsrq_attention_decode;
    calls that overlap on one GPU race on the shared buffer (include/gsrq.h)."""
    Bq, Hq, hd = q.shape
    _check(lib().gsrq_attention_decode_static(_ptr(q), _ptr(k_codes), C.byref(k_cb), k_stages, _ptr(v_codes), C.byref(v_cb), v_stages,
                                              C.c_int64(plane_rows), _ptr(seq_start), _ptr(seq_len), C.c_int64(max_len), Bq, Hq, G, hd, d,
                                              C.c_float(scale), C.c_float(rope_theta), _ptr(out), _stream()))


def gsrq_log_weights(grad, view, tau, eps, w_out):
    _check(lib().gsrq_log_weights(_ptr(grad), C.byref(view), C.c_float(tau), C.c_float(eps), _ptr(w_out), _stream()))


def gsrq_encode_pervector_gain(kv, view, cb, n_stages, codes, gains16, residual, ws):
    _check(lib().gsrq_encode_pervector_gain(_ptr(kv), C.byref(view), C.byref(cb), n_stages, _ptr(codes), _ptr(gains16), _ptr(residual),
                                            _ptr(ws), C.c_size_t(ws.numel()), _stream()))


def gsrq_decode_pervector_gain(codes, gains16, cb, n_stages, kv_out, out_view):
    _check(lib().gsrq_decode_pervector_gain(_ptr(codes), _ptr(gains16), C.byref(cb), n_stages, _ptr(kv_out), C.byref(out_view), _stream()))


def gsrq_pack_nibbles(codes, K, n_planes, N, packed):
    _check(lib().gsrq_pack_nibbles(_ptr(codes), K, C.c_int64(n_planes), C.c_int64(N), _ptr(packed), _stream()))


def gsrq_unpack_nibbles(packed, n_planes, N, codes):
    _check(lib().gsrq_unpack_nibbles(_ptr(packed), C.c_int64(n_planes), C.c_int64(N), _ptr(codes), _stream()))


def cluster_workspace(N: int, d: int, K: int) -> torch.Tensor:
    n = lib().gsrq_cluster_workspace_bytes(C.c_int64(N), d, K)
    if n == 0:
        raise GsrqError(-1, lib().gsrq_last_error().decode())
    return torch.empty(n, dtype=torch.uint8, device="cuda")


def gsrq_cluster_fit(x, w, K, iters, seed, method, shapes, gains, idx_out, ws, want_stats=True):
    """x [N][d] fp32 CUDA rows; method 0 = GSKM, 1 = K-means; shapes [K][d], gains [K] fp32, idx_out [N] int16/uint16 storage."""
    N, d = x.shape
    stats = (gsrq_fit_stats * 1)() if want_stats else None
    _check(lib().gsrq_cluster_fit(_ptr(x), _ptr(w), C.c_int64(N), d, K, iters, C.c_uint64(seed), method, _ptr(shapes), _ptr(gains),
                                  _ptr(idx_out), stats, _ptr(ws), C.c_size_t(ws.numel()), _stream()))
    return stats


def gsrq_cluster_assign(x, K, method, shapes, gains, idx_out):
    N, d = x.shape
    _check(lib().gsrq_cluster_assign(_ptr(x), C.c_int64(N), d, K, method, _ptr(shapes), _ptr(gains), _ptr(idx_out), _stream()))


def gsrq_cluster_metrics(x, K, method, shapes, gains, idx, ws):
    """Returns dict(mse, gain_err, cosine, shrinkage) of the reconstruction by the assigned prototypes."""
    N, d = x.shape
    out = (C.c_double * 4)()
    _check(lib().gsrq_cluster_metrics(_ptr(x), C.c_int64(N), d, K, method, _ptr(shapes), _ptr(gains), _ptr(idx), out, _ptr(ws),
                                      C.c_size_t(ws.numel()), _stream()))
    return dict(mse=out[0], gain_err=out[1], cosine=out[2], shrinkage=out[3])


def gsrq_encode_host(kv_host: torch.Tensor, view, cb, codes_host: torch.Tensor):
    """kv_host / codes_host are HOST tensors (pinned or pageable); copies happen inside the call."""
    assert not kv_host.is_cuda and not codes_host.is_cuda
    _check(lib().gsrq_encode_host(_ptr(kv_host), C.byref(view), C.byref(cb), _ptr(codes_host)))


def gsrq_decode_host(codes_host: torch.Tensor, cb, n_stages, kv_out_host: torch.Tensor, out_view):
    assert not kv_out_host.is_cuda and not codes_host.is_cuda
    _check(lib().gsrq_decode_host(_ptr(codes_host), C.byref(cb), n_stages, _ptr(kv_out_host), C.byref(out_view)))


def gsrq_pipeline_host(kv_host, view, w_host, fit_tokens_host, K, S, iters, seed, shapes_host, gains_host, codes_host, kv_out_host):
    """All arguments are HOST tensors; H2D, fit + encode (+ decode), D2H and the sync happen inside."""
    for t in (kv_host, w_host, fit_tokens_host, shapes_host, gains_host, codes_host, kv_out_host):
        assert t is None or not t.is_cuda
    n_fit = 0 if fit_tokens_host is None else fit_tokens_host.shape[1]
    _check(lib().gsrq_pipeline_host(_ptr(kv_host), C.byref(view), _ptr(w_host), _ptr(fit_tokens_host), C.c_int64(n_fit), K, S, iters,
                                    C.c_uint64(seed), _ptr(shapes_host), _ptr(gains_host), _ptr(codes_host), _ptr(kv_out_host)))


def gsrq_pipeline_host_batch(kv_hosts, view, w_hosts, fit_tokens_hosts, K, S, iters, seed, shapes_hosts, gains_hosts, codes_hosts, kv_out_hosts):
    """gsrq_pipeline_host for a list of HOST tensors of the same view (e.g. a layer's K and V cache), pipelined over two streams.
    w_hosts / fit_tokens_hosts / kv_out_hosts: lists (entries may be None) or None."""
    n = len(kv_hosts)
    def arr(ts):
        if ts is None:
            return None
        assert len(ts) == n
        for t in ts:
            assert t is None or not t.is_cuda
        return (C.c_void_p * n)(*[(t.data_ptr() if t is not None else None) for t in ts])
    n_fit = 0
    if fit_tokens_hosts is not None:
        shp = {t.shape[1] for t in fit_tokens_hosts if t is not None}
        assert len(shp) <= 1, "the tensors of a batch share n_fit"
        n_fit = shp.pop() if shp else 0
    _check(lib().gsrq_pipeline_host_batch(n, arr(kv_hosts), C.byref(view), arr(w_hosts), arr(fit_tokens_hosts), C.c_int64(n_fit), K, S, iters,
                                          C.c_uint64(seed), arr(shapes_hosts), arr(gains_hosts), arr(codes_hosts), arr(kv_out_hosts)))


def gsrq_release_host_pool():
    lib().gsrq_release_host_pool()


KERNEL_CLASSES = ["prep", "score", "refine", "update", "misc", "decode", "encode"]


def gsrq_profile_enable(on: bool):
    lib().gsrq_profile_enable(int(on))


def gsrq_profile_read():
    """Per kernel class: (summed device ms, launches) since the last read."""
    ms = (C.c_double * len(KERNEL_CLASSES))()
    n = (C.c_int64 * len(KERNEL_CLASSES))()
    _check(lib().gsrq_profile_read(ms, n))
    return {k: (ms[i], n[i]) for i, k in enumerate(KERNEL_CLASSES)}


def gsrq_launch_count() -> int:
    return int(lib().gsrq_launch_count())
