"""attn_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain fp64 definition of the decoding step the paper fuses with dequantisation (PAPER.md:443 (ii): "on-the-fly bit-unpacking,
dequantization, RoPE, and attention computation during decoding without materializing intermediate FP16 tensors"): for every
sequence b and query head h of the new token,

    khat_t = sum_s cK^(s)[aK^(s)_t]      (fp32 sums in stage order exactly as gsrq_decode, reading c-D, NOT cast to bf16)
    vhat_t = sum_s cV^(s)[aV^(s)_t]
    k_t    = RoPE(khat_t, position t)     (optional: the keys are quantised before the rotary embedding)
    out_h  = sum_t softmax_t(scale * q_h . k_t) vhat_t      over the tokens t of sequence b, KV head g = h // (Hq / G)

Readings (the paper gives no formula for this step): rotary embedding in the "rotate-half" convention of the LLaMA family the
paper evaluates -- element i < hd/2 pairs with i + hd/2, angle = position * theta^(-2 i / hd); the query is given already
rotated; grouped-query attention maps query head h to KV head h // (Hq / G) (LLaMA-3-8B: 32 query heads, 8 KV heads,
PAPER.md:216); scale = 1/sqrt(hd) unless given.  Everything after the fp32 decode is numpy float64.  It imports nothing from
the CUDA path.
"""
from __future__ import annotations

import numpy as np

from . import gsrq_oracle as o


def rope(x, pos, theta):
    """Rotate-half rotary embedding of x [..., hd] (float64) at integer positions pos [...]."""
    hd = x.shape[-1]
    half = hd // 2
    inv = theta ** (-np.arange(half, dtype=np.float64) * 2.0 / hd)
    ang = np.asarray(pos, dtype=np.float64)[..., None] * inv
    c, s = np.cos(ang), np.sin(ang)
    a, b = x[..., :half], x[..., half:]
    return np.concatenate([a * c - b * s, b * c + a * s], axis=-1)


def decode_f32(codes, shapes, gains, hd):
    """codes [S][G][Ng] -> [G][T][hd] fp32 (stage-order fp32 sums, no bf16 cast)."""
    out, _ = o.decode(codes, shapes, gains, hd, bf16=False)
    return out


def attention_decode(q, k_codes, k_shapes, k_gains, v_codes, v_shapes, v_gains, hd, seq_start, seq_len, scale=None, rope_theta=0.0):
    """q [B][Hq][hd]; codes [S][G][Tc*M]; returns out [B][Hq][hd] float64 (zeros for an empty sequence)."""
    q = np.asarray(q, dtype=np.float64)
    B, Hq, _ = q.shape
    G = k_codes.shape[1]
    n_rep = Hq // G
    scale = 1.0 / np.sqrt(hd) if scale is None else scale
    khat = decode_f32(k_codes, k_shapes, k_gains, hd).astype(np.float64)   # [G][Tc][hd]
    vhat = decode_f32(v_codes, v_shapes, v_gains, hd).astype(np.float64)
    out = np.zeros((B, Hq, hd), dtype=np.float64)
    for b in range(B):
        t0, n = int(seq_start[b]), int(seq_len[b])
        if n == 0:
            continue
        for h in range(Hq):
            g = h // n_rep
            k = khat[g, t0:t0 + n]
            if rope_theta > 0.0:
                k = rope(k, np.arange(n), rope_theta)
            logits = scale * (k @ q[b, h])
            p = np.exp(logits - logits.max())
            p /= p.sum()
            out[b, h] = p @ vhat[g, t0:t0 + n]
    return out
