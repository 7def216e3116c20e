"""Seeded random shapes through the whole GPU path (fit -> encode -> decode) against the oracle: every
combination of sub-vector dimension, head_dim, K, S, layout, dtype, weights and fit subset that the library
accepts, at sizes the oracle finishes in a fraction of a second.  BASELINE.json's criteria (a)(b)(c)."""
import numpy as np
import pytest

from paper_2607_01065_b200.pipeline import gpu_decode, gpu_gsrq
from oracle import gsrq_oracle as o
from paper_2607_01065_b200 import inputs

pytestmark = pytest.mark.gpu


def _case(seed, wide=False):
    rng = np.random.default_rng(1000 + seed)
    d = int(rng.choice([64, 128, 128, 256])) if wide else int(rng.choice([8, 16, 16, 16, 32]))
    M = int(rng.choice([1, 1, 2])) if wide else int(rng.choice([1, 2, 4, 8]))
    hd = d * M
    G = int(rng.integers(1, 5))
    T = int(rng.integers(40, 400))
    K = int(rng.choice([1, 7, 16, 100, 256]))
    K = min(K, max(1, (T * M) // 3))
    S = int(rng.integers(1, 4 if wide else 5))
    iters = int(rng.integers(0, 5 if wide else 6))
    dtype = "bf16" if rng.random() < 0.7 else "f32"
    head_inner = bool(rng.random() < 0.4)
    x = rng.standard_normal((G, T, hd)) * np.exp(0.6 * rng.standard_normal((G, T, 1)))
    if rng.random() < 0.3:
        x[:, rng.integers(0, T, 3)] = 0.0                       # a few all-zero tokens
    x = inputs.bf16_round(x) if dtype == "bf16" else x.astype(np.float32)
    w = None if rng.random() < 0.3 else (np.exp(rng.standard_normal(T)) / 1.6).astype(np.float32)
    fit = None
    if rng.random() < 0.4 and T >= 120:
        n_fit = int(rng.integers(max(K // M + 8, 30), T))
        fit = inputs.fit_sample(G, T, n_fit, 77 + seed)
    return dict(x=x, w=w, d=d, hd=hd, K=K, S=S, iters=iters, dtype=dtype, head_inner=head_inner, fit=fit,
                pass_residual=bool(rng.random() < 0.5), prefix=bool(rng.random() < 0.5))


@pytest.mark.parametrize("seed", list(range(16)) + [100 + i for i in range(8)])
def test_random_shapes_match_oracle(seed):
    c = _case(seed, wide=seed >= 100)   # seeds >= 100: the wide sub-vectors d = 64 / 128 / 256 (tcgen05 filter / exact fp64 kernels)
    x, w, d, K, S = c["x"], c["w"], c["d"], c["K"], c["S"]
    G, T, hd = x.shape
    M = hd // d
    try:
        ref = o.gsrq_fit_encode(x, w, d, K, S, c["iters"], seed=seed, fit_tokens=c["fit"])
    except ValueError:
        pytest.skip("degenerate draw (fewer than K distinct non-zero rows)")
    got = gpu_gsrq(x, w, d, K, S, c["iters"], seed=seed, dtype=c["dtype"], fit_tokens=c["fit"], head_inner=c["head_inner"],
                   pass_residual=c["pass_residual"] and c["fit"] is None, prefix_encode=c["prefix"])
    assert np.abs(got["shapes"] - ref["shapes"]).max() <= 1e-4, c
    assert np.abs(got["gains"] - ref["gains"]).max() <= 1e-4, c
    r = o.rows_of(x, d).copy()
    bad = 0
    for st in range(S):
        n_st = np.linalg.norm(r.astype(np.float64), axis=-1)
        gap = ref["best"][st] - ref["second"][st]
        bad += int(((got["codes"][st] != ref["codes"][st]) & (gap >= 1e-5 * n_st)).sum())
        for g_ in range(G):
            _, r[g_], _, _ = o.encode_stage(r[g_], ref["shapes"][g_, st], ref["gains"][g_, st])
    assert bad == 0, c
    w_rows = np.ones(T * M) if w is None else np.repeat(w, M).astype(np.float64)
    for g_ in range(G):
        jr = float((w_rows * (ref["residual"][g_].astype(np.float64) ** 2).sum(-1)).sum())
        jg = float((w_rows * (got["residual"][g_].astype(np.float64) ** 2).sum(-1)).sum())
        assert abs(jr - jg) <= 1e-4 * max(jr, 1e-30), c
    dec = gpu_decode(got["codes_dev"], got["cb"], S, G, T, hd, d, dtype=c["dtype"], head_inner=c["head_inner"])
    want, _ = o.decode(got["codes"], got["shapes"], got["gains"], hd, bf16=(c["dtype"] == "bf16"))
    assert np.array_equal(dec, want), c
