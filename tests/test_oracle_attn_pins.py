"""Pins of oracle/attn_oracle.py (the decode-attention step of PAPER.md:443 (ii)) against a library routine and the closed-form
properties of the rotary embedding.  CPU only."""
import numpy as np
import pytest
import torch

from oracle import attn_oracle as ao
from oracle import gsrq_oracle as o


def _setup(G=2, Tc=96, hd=32, d=8, K=16, S=2, seed=0):
    rng = np.random.default_rng(seed)
    M = hd // d
    def cb():
        s = rng.standard_normal((G, S, K, d)); s /= np.linalg.norm(s, axis=-1, keepdims=True)
        return s.astype(np.float32), np.abs(rng.standard_normal((G, S, K))).astype(np.float32)
    ks, kg = cb(); vs, vg = cb()
    kc = rng.integers(0, K, (S, G, Tc * M)).astype(np.uint8)
    vc = rng.integers(0, K, (S, G, Tc * M)).astype(np.uint8)
    return dict(ks=ks, kg=kg, vs=vs, vg=vg, kc=kc, vc=vc, hd=hd, G=G, Tc=Tc)


def test_attention_matches_torch_sdpa_on_the_decoded_tensors():
    c = _setup()
    B, Hq = 3, 4
    rng = np.random.default_rng(1)
    q = rng.standard_normal((B, Hq, c["hd"]))
    start, length = np.array([0, 10, 50]), np.array([10, 40, 46])
    out = ao.attention_decode(q, c["kc"], c["ks"], c["kg"], c["vc"], c["vs"], c["vg"], c["hd"], start, length)
    khat = torch.from_numpy(ao.decode_f32(c["kc"], c["ks"], c["kg"], c["hd"])).double()
    vhat = torch.from_numpy(ao.decode_f32(c["vc"], c["vs"], c["vg"], c["hd"])).double()
    for b in range(B):
        for h in range(Hq):
            g = h // (Hq // c["G"])
            k = khat[g, start[b]:start[b] + length[b]][None, None]
            v = vhat[g, start[b]:start[b] + length[b]][None, None]
            want = torch.nn.functional.scaled_dot_product_attention(torch.from_numpy(q[b, h])[None, None, None], k, v)[0, 0, 0]
            np.testing.assert_allclose(out[b, h], want.numpy(), rtol=1e-10, atol=1e-12)


def test_decode_is_the_stage_order_sum_of_scaled_codewords():
    c = _setup(S=3)
    khat = ao.decode_f32(c["kc"], c["ks"], c["kg"], c["hd"])
    g, t, m, d = 1, 17, 2, 8
    want = np.float32(0)
    acc = None
    for s in range(3):
        k = c["kc"][s, g, t * 4 + m]
        cw = (c["kg"][g, s, k] * c["ks"][g, s, k]).astype(np.float32)
        acc = cw if acc is None else (acc + cw).astype(np.float32)
    assert np.array_equal(khat[g, t, m * d:(m + 1) * d], acc)


def test_rope_properties():
    rng = np.random.default_rng(2)
    x, y = rng.standard_normal((5, 64)), rng.standard_normal((5, 64))
    # position 0 is the identity; norms are preserved; <R_m x, R_n y> depends on m - n only
    assert np.array_equal(ao.rope(x, np.zeros(5), 10000.0), x)
    np.testing.assert_allclose(np.linalg.norm(ao.rope(x, np.arange(5) * 37, 10000.0), axis=-1), np.linalg.norm(x, axis=-1), rtol=1e-12)
    a = (ao.rope(x, np.full(5, 100), 10000.0) * ao.rope(y, np.full(5, 93), 10000.0)).sum(-1)
    b = (ao.rope(x, np.full(5, 7), 10000.0) * y).sum(-1)
    np.testing.assert_allclose(a, b, rtol=1e-9)
    # first frequency is theta^0 = 1: the pair (x_0, x_{hd/2}) rotates by exactly `position` radians
    e = np.zeros((1, 64)); e[0, 0] = 1.0
    r = ao.rope(e, np.array([0.5]), 10000.0)
    assert r[0, 0] == pytest.approx(np.cos(0.5)) and r[0, 32] == pytest.approx(np.sin(0.5))


def test_rope_attention_equals_attention_on_rotated_keys_and_empty_sequence():
    c = _setup(seed=3)
    q = np.random.default_rng(4).standard_normal((2, 2, c["hd"]))
    start, length = np.array([5, 0]), np.array([30, 0])
    out = ao.attention_decode(q, c["kc"], c["ks"], c["kg"], c["vc"], c["vs"], c["vg"], c["hd"], start, length, rope_theta=500.0)
    khat = ao.decode_f32(c["kc"], c["ks"], c["kg"], c["hd"]).astype(np.float64)
    vhat = ao.decode_f32(c["vc"], c["vs"], c["vg"], c["hd"]).astype(np.float64)
    k = ao.rope(khat[1, 5:35], np.arange(30), 500.0)
    lg = (k @ q[0, 1]) / np.sqrt(c["hd"])
    p = np.exp(lg - lg.max()); p /= p.sum()
    np.testing.assert_allclose(out[0, 1], p @ vhat[1, 5:35], rtol=1e-12)
    assert not out[1].any()
