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


def test_rope_frequency_schedule_hand_values():
    """Pins the inverse frequencies of ao.rope for i >= 1 (reading a-R of DESIGN.md: rotate-half convention of the LLaMA family,
    angle_i = position * theta^(-2 i / hd)).  Hand values for hd = 8, theta = 10000, position 3: pair (i, i + 4) turns by
    3 * 10000^(-2 i / 8) = 3, 0.3, 0.03, 0.003 radians for i = 0..3.  A schedule of theta^(-i / hd) (angles 3, 0.949, 0.3, 0.0949)
    or any other exponent fails."""
    x = np.array([[1.0, 2.0, -3.0, 0.5, 0.25, -1.5, 4.0, 2.5]])
    r = ao.rope(x, np.array([3]), 10000.0)[0]
    for i, ang in enumerate([3.0, 0.3, 0.03, 0.003]):
        a, b = x[0, i], x[0, i + 4]
        assert r[i] == pytest.approx(a * np.cos(ang) - b * np.sin(ang), rel=1e-12, abs=1e-14), i
        assert r[i + 4] == pytest.approx(b * np.cos(ang) + a * np.sin(ang), rel=1e-12, abs=1e-14), i
    # literal numbers (cos / sin of 0.3 and 0.03 typed in, not computed): element 1 and 5, element 2 and 6
    assert r[1] == pytest.approx(2.0 * 0.955336489125606 + 1.5 * 0.29552020666133955, rel=1e-12)
    assert r[5] == pytest.approx(-1.5 * 0.955336489125606 + 2.0 * 0.29552020666133955, rel=1e-12)
    assert r[2] == pytest.approx(-3.0 * 0.9995500337489875 - 4.0 * 0.02999550020249566, rel=1e-12)
    assert r[6] == pytest.approx(4.0 * 0.9995500337489875 - 3.0 * 0.02999550020249566, rel=1e-12)


def test_rope_equals_the_llama_rotary_embedding_of_transformers():
    """The same pin against a library: transformers' LLaMA rotary embedding (inverse frequencies and apply_rotary_pos_emb's
    rotate-half pairing) at LLaMA-3's head_dim 128 / theta 500000 (the model family of PAPER.md:216)."""
    pytest.importorskip("transformers")
    from transformers import LlamaConfig
    from transformers.models.llama.modeling_llama import LlamaRotaryEmbedding, apply_rotary_pos_emb
    hd, nh, theta = 128, 2, 500000.0
    rot = LlamaRotaryEmbedding(config=LlamaConfig(hidden_size=hd * nh, num_attention_heads=nh, num_key_value_heads=nh, rope_theta=theta,
                                                  max_position_embeddings=4096))
    # the oracle's inverse frequencies, read off its output: e_i at position 1 turns by inv_i
    eye = np.eye(hd)[: hd // 2]
    r = ao.rope(eye, np.ones(hd // 2), theta)
    inv = np.arctan2(r[np.arange(hd // 2), np.arange(hd // 2) + hd // 2], r[np.arange(hd // 2), np.arange(hd // 2)])
    np.testing.assert_allclose(inv, rot.inv_freq.double().numpy(), rtol=2e-6)   # the library stores them in fp32
    x = torch.randn(1, nh, 4, hd, dtype=torch.float64, generator=torch.Generator().manual_seed(5))
    pos = torch.tensor([[0, 1, 7, 100]])
    cos, sin = rot(x, pos)
    want, _ = apply_rotary_pos_emb(x, x, cos.double(), sin.double())
    got = ao.rope(x[0].numpy(), np.broadcast_to(pos.numpy(), (nh, 4)), theta)
    np.testing.assert_allclose(got, want[0].numpy(), atol=2e-5)
