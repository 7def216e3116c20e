"""Pins of oracle/variants_oracle.py against closed forms, the paper's own statements and hand-written examples.  CPU only."""
import numpy as np
import pytest

from oracle import gsrq_oracle as o
from oracle import variants_oracle as vo


def test_log_weights_closed_forms_and_the_papers_dynamic_range_statement():
    rng = np.random.default_rng(0)
    g = rng.standard_normal((2, 301, 16)) * np.exp(rng.standard_normal((2, 301, 1)))
    w = vo.log_weights(g, tau=1.0, eps=0.0)
    nrm = np.sqrt((g ** 2).sum(-1)).astype(np.float32).astype(np.float64)
    med = np.median(nrm, axis=-1)
    # the token at the median maps to log(1 + tau) (Eq. 10: the median is scaled to tau before log(1 + x))
    for h in range(2):
        i = int(np.argsort(nrm[h])[150])
        assert w[h, i] == pytest.approx(np.log(2.0), rel=1e-6)
        assert (np.diff(w[h][np.argsort(nrm[h])]) >= 0).all()            # monotone in ||g||
        np.testing.assert_allclose(w[h], np.log(1.0 + nrm[h] / med[h]), rtol=1e-6)
    # raw norms with max / median > 400x are compressed to a ratio below 10x (tau = 1): log(401) / log(2) = 8.65
    raw = np.ones((1, 101, 1)); raw[0, 0, 0] = 400.0
    t = vo.log_weights(raw, tau=1.0, eps=0.0)
    assert t[0].max() / np.median(t[0]) == pytest.approx(np.log(401.0) / np.log(2.0), rel=1e-6) and t[0].max() / np.median(t[0]) < 10.0
    # even count: numpy's median is the mean of the two middle values
    ev = np.array([[[1.0], [2.0], [4.0], [100.0]]])
    np.testing.assert_allclose(vo.log_weights(ev, tau=3.0, eps=0.0)[0], np.log1p(3.0 / 3.0 * np.array([1.0, 2.0, 4.0, 100.0])), rtol=1e-6)


def test_pervector_gain_is_the_clamped_projection_rounded_to_fp16():
    rng = np.random.default_rng(1)
    r = (rng.standard_normal((500, 16)) * np.exp(0.5 * rng.standard_normal((500, 1)))).astype(np.float32)
    s = rng.standard_normal((32, 16)); s = (s / np.linalg.norm(s, axis=1, keepdims=True)).astype(np.float32)
    codes, gam, res = vo.encode_stage_pervector_gain(r, s)
    proj = r.astype(np.float64) @ s.astype(np.float64).T
    assert np.array_equal(codes, proj.argmax(1))
    np.testing.assert_array_equal(gam, np.maximum(proj.max(1), 0).astype(np.float16))
    # the residual is (nearly) orthogonal to the chosen shape: |res . s_k| <= fp16 rounding of gamma (2^-11 gamma) + fp32 noise
    dot = (res.astype(np.float64) * s[codes].astype(np.float64)).sum(1)
    assert (np.abs(dot) <= 2.0 ** -11 * gam.astype(np.float64) + 1e-5).all()
    assert (np.linalg.norm(res, axis=1) <= np.linalg.norm(r, axis=1) * (1 + 1e-6)).all()      # projection never lengthens
    # reconstruction + residual = x to fp32 rounding; a second stage decodes in stage order
    codes2, gam2, res2 = vo.encode_stage_pervector_gain(res, s)
    xhat = vo.decode_pervector_gain(np.stack([codes, codes2]), np.stack([gam, gam2]), np.stack([s, s]))
    np.testing.assert_allclose(xhat + res2, r, atol=1e-5)
    # a row whose projections are all negative gets gain 0 (clamp) and an untouched residual
    pos = np.abs(s[:4]) / np.linalg.norm(np.abs(s[:4]), axis=1, keepdims=True)
    row = -np.ones((1, 16), np.float32)
    _, g0, r0 = vo.encode_stage_pervector_gain(row, pos.astype(np.float32))
    assert g0[0] == 0 and np.array_equal(r0, row)


def test_nibble_packing_hand_example_and_round_trip():
    assert np.array_equal(vo.pack_nibbles(np.array([1, 2, 15, 0, 7], np.uint8)), np.array([0x21, 0x0F, 0x07], np.uint8))
    rng = np.random.default_rng(2)
    c = rng.integers(0, 16, (2, 3, 1001)).astype(np.uint8)
    p = vo.pack_nibbles(c)
    assert p.shape == (2, 3, 501) and np.array_equal(vo.unpack_nibbles(p, 1001), c)
