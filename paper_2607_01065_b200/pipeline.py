"""Convenience drivers over the C-ABI binding (argument marshalling and call sequencing only; every step runs in libgsrq):
fit the stages one after the other with the fused prefix encode in between, and decode.  Used by the tests,
__graft_entry__.smoke() and as the shortest example of the call sequence."""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B


def to_device(x_np: np.ndarray, dtype: str, head_inner: bool = False) -> torch.Tensor:
    """x_np [G][T][hd] fp32 values -> CUDA tensor of the storage dtype ([T][G][hd] memory if head_inner)."""
    t = torch.from_numpy(np.ascontiguousarray(x_np))
    if head_inner:
        t = t.permute(1, 0, 2).contiguous()
    t = t.to(torch.bfloat16 if dtype == "bf16" else torch.float32)
    return t.cuda()


def gpu_gsrq(x_np, w_np, d, K, S, iters, seed=0, dtype="bf16", fit_tokens=None, head_inner=False,
             pass_residual=True, want_residual=True, prefix_encode=False):
    """fit stage by stage + encode on the GPU. Returns numpy results + stats.
    pass_residual: each stage is encoded right after its fit and its residual feeds the next fit
    (prefix_encode: that encode is the fused [0, s] pass, as bench.py does; else stage s alone);
    otherwise the fits re-derive their residual and one fused encode of all stages follows."""
    x = to_device(x_np, dtype, head_inner)
    view = B.view_of(x, d, head_inner)
    G, T, hd = view.G, view.T, view.hd
    M = hd // d
    w = None if w_np is None else torch.from_numpy(np.ascontiguousarray(w_np, dtype=np.float32)).cuda()
    w_stride = 0 if (w is None or w.dim() == 1) else w.stride(0)
    ft = None if fit_tokens is None else torch.from_numpy(np.ascontiguousarray(fit_tokens, dtype=np.int64)).cuda()
    shapes = torch.zeros(G, S, K, d, dtype=torch.float32, device="cuda")
    gains = torch.zeros(G, S, K, dtype=torch.float32, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, S, 0)
    codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
    residual = torch.zeros(G, T * M, d, dtype=torch.float32, device="cuda")
    stats = []
    for st in range(S):
        res_in = residual if (pass_residual and st > 0) else None
        s = B.gsrq_fit_stage(x, view, w, w_stride, ft, cb, st, res_in, iters, seed, ws)
        stats.append(s)
        if pass_residual:
            B.gsrq_encode(x, view, cb, 0 if prefix_encode else st, st + 1, codes, residual, ws)
    if not pass_residual:
        B.gsrq_encode(x, view, cb, 0, S, codes, residual if want_residual else None, ws)
    torch.cuda.synchronize()
    return dict(shapes=shapes.cpu().numpy(), gains=gains.cpu().numpy(), codes=codes.cpu().numpy(),
                residual=residual.cpu().numpy(), stats=stats, x=x, view=view, cb=cb, ws=ws,
                codes_dev=codes, shapes_dev=shapes, gains_dev=gains)


def stats_np(stats, g):
    s = stats[g]
    n = s.iters_run
    return dict(iters_run=n, n_empty_last=s.n_empty_last, n_changed_last=s.n_changed_last, n_refined=s.n_refined,
                J=np.array(s.wdist_after_assign[:n]), changed=np.array(s.n_changed[:n]))


def gpu_decode(codes_dev, cb, n_stages, G, T, hd, d, dtype="bf16", head_inner=False):
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    out = torch.zeros((T, G, hd) if head_inner else (G, T, hd), dtype=tdt, device="cuda")
    B.gsrq_decode(codes_dev, cb, n_stages, out, B.view_of(out, d, head_inner))
    torch.cuda.synchronize()
    o = out.permute(1, 0, 2) if head_inner else out
    return o.float().cpu().numpy()
