"""variants_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy definitions of the small variants around the GSRQ encoder, each written from the passage it
cites; nothing here is imported by the CUDA path.

* Log-smoothed gradient weights (PAPER.md:192 Eq. 9; :434 Eq. 10):  w = ||g||_2 per token,  lambda = tau / (median(w) + eps),
  w~ = log(1 + lambda w).  Double precision; the median is numpy's (mean of the two middle values for an even count).
* Per-vector gain codes (the alternative reading c-G of "a codeword index plus a gain", BASELINE.json config 0 "4-bit indices plus an
  fp16 gain"): shape-gain coding of one RQ stage -- k = argmax_k r.s_k (lowest k on ties), gamma = fp16(max(0, r.s_k)) (dot product
  in double, one round-to-nearest-even cast), r <- fl32(r - fl32(fl32(gamma) s_k)); decode sums fl32(gamma s_k) in fp32 stage order.
  The codebook's shapes come from GSKM as usual; its per-cluster gains are not used.  Costs 16/d extra bits per element per stage.
* Nibble packing for K <= 16 (BASELINE.json config 0 "Codes are 4-bit indices"; "bit-packing"): two codes per byte,
  row 2i in the low nibble, row 2i+1 in the high nibble; an odd last row leaves the high nibble 0.
* Per-subspace codebooks ("an independent codebook per subspace"): subspace m of head g is the tensor x[g][:, m d:(m+1) d]
  quantised on its own, i.e. the ordinary encoder on a [G][T][d] view.
"""
from __future__ import annotations

import numpy as np

from . import gsrq_oracle as o


def log_weights(grad, tau=1.0, eps=1e-12):
    """grad [G][T][hd] -> w~ [G][T] float32 (Eq. 9-10), per head."""
    w = np.sqrt((np.asarray(grad, dtype=np.float64) ** 2).sum(-1)).astype(np.float32).astype(np.float64)   # the norm is stored as fp32
    lam = tau / (np.median(w, axis=-1, keepdims=True) + eps)
    return np.log1p(lam * w).astype(np.float32)


def encode_stage_pervector_gain(r, s):
    """One shape-gain stage on rows r [N][d] with unit shapes s [K][d]. Returns codes u8, gains fp16, new residual fp32."""
    r = np.ascontiguousarray(r, dtype=np.float32)
    s = np.ascontiguousarray(s, dtype=np.float32)
    idx, best, _ = o.assign(r, s, None)                  # plain projection arg-max in double, lowest k on ties
    gamma = np.maximum(best, 0.0).astype(np.float16)     # one RN-even cast from double
    c = (gamma.astype(np.float32)[:, None] * s[idx]).astype(np.float32)
    return idx.astype(np.uint8), gamma, (r - c).astype(np.float32)


def decode_pervector_gain(codes, gains16, shapes):
    """codes [S][N], gains16 [S][N] fp16, shapes [S][K][d] -> xhat [N][d] fp32 (stage-order fp32 sum)."""
    acc = None
    for st in range(codes.shape[0]):
        c = (gains16[st].astype(np.float32)[:, None] * shapes[st][codes[st]]).astype(np.float32)
        acc = c if acc is None else (acc + c).astype(np.float32)
    return acc


def pack_nibbles(codes):
    """codes [..., N] uint8 (< 16) -> [..., ceil(N/2)] uint8."""
    codes = np.asarray(codes, dtype=np.uint8)
    N = codes.shape[-1]
    pad = np.zeros(codes.shape[:-1] + (N + (N & 1),), dtype=np.uint8)
    pad[..., :N] = codes
    return (pad[..., 0::2] | (pad[..., 1::2] << 4)).astype(np.uint8)


def unpack_nibbles(packed, N):
    out = np.zeros(packed.shape[:-1] + (2 * packed.shape[-1],), dtype=np.uint8)
    out[..., 0::2] = packed & 15
    out[..., 1::2] = packed >> 4
    return out[..., :N]
