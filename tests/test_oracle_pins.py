"""Pins for the CPU oracle (oracle/gsrq_oracle.c).  CPU only.

Each test checks the oracle against something OTHER than itself: brute force, a closed
form, an invariant fixed by the paper's equations, a textbook / scikit-learn routine the
method reduces to in a special case, or a cited golden value.
"""
import math
from pathlib import Path

import numpy as np
import pytest

from oracle import gsrq_oracle as o
from paper_2607_01065_b200 import inputs

GOLD = Path(__file__).parent / "golden"


def _unit(v):
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _rand_codebook(rng, K, d):
    s = _unit(rng.standard_normal((K, d))).astype(np.float32)
    g = np.abs(rng.standard_normal(K)).astype(np.float32) * 2
    return s, g


# ---------------------------------------------------------------- generator pin
def test_splitmix64_published_vectors():
    for line in (GOLD / "splitmix64.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        seed, n, val = line.split()
        got = o.splitmix64(int(seed), int(n) + 1)[int(n)]
        assert got == int(val, 0)


def test_init_ids_follow_reading_c_I():
    """Re-derive the candidate stream in pure Python ints (independent of the C code)."""
    rng = np.random.default_rng(5)
    r = rng.standard_normal((50, 4)).astype(np.float32)
    r[[3, 7, 11, 20]] = 0.0                     # zero rows must be rejected
    K, seed, group, G, stage = 16, 0, 2, 8, 1
    mask = (1 << 64) - 1
    st = seed ^ ((0x9E3779B97F4A7C15 * (1 + group + G * stage)) & mask)
    want = []
    while len(want) < K:
        st = (st + 0x9E3779B97F4A7C15) & mask
        z = st
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & mask
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & mask
        z ^= z >> 31
        c = z % 50
        if c in want or not r[c].any():
            continue
        want.append(c)
    got = o.init_ids(r, K, seed, group, G, stage)
    assert got.tolist() == want
    assert len(set(got.tolist())) == K
    with pytest.raises(ValueError):
        o.init_ids(np.zeros((50, 4), np.float32), K, 0)


# ---------------------------------------------------------------- assignment (Eq. 4, 5)
def test_assignment_is_brute_force_nearest_centroid():
    rng = np.random.default_rng(0)
    for d, K, N in [(2, 3, 200), (8, 16, 500), (16, 256, 300)]:
        x = (rng.standard_normal((N, d)) * np.exp(0.5 * rng.standard_normal((N, 1)))).astype(np.float32)
        s, g = _rand_codebook(rng, K, d)
        g[rng.integers(K)] = 0.0                # a zero-gain cluster (reconstruction 0) is legal
        idx, best, second = o.assign(x, s, g)
        mu = g[:, None].astype(np.float64) * s.astype(np.float64)
        d2 = ((x[:, None, :].astype(np.float64) - mu[None]) ** 2).sum(-1)      # direct ||x - g s||^2
        assert np.array_equal(idx, d2.argmin(1))
        # Eq. 4: ||x - g s||^2 = ||x||^2 + g^2 - 2 g x.s  (with ||s|| = 1 up to fp32 rounding of s)
        n2 = (x.astype(np.float64) ** 2).sum(1)
        snorm2 = (s.astype(np.float64) ** 2).sum(1)
        corr = (g.astype(np.float64) ** 2 * (snorm2 - 1.0))[idx]               # exact-unit-norm correction
        np.testing.assert_allclose(n2 - best + corr, d2.min(1), rtol=0, atol=1e-9 * (1 + n2.max()))
        assert (second <= best).all()


def test_assignment_ties_go_to_lowest_index_and_projection_mode():
    s = np.array([[1, 0], [1, 0], [0, 1]], np.float32)
    g = np.array([1, 1, 1], np.float32)
    x = np.array([[2, 0], [0, 3], [1, 1]], np.float32)
    idx, best, second = o.assign(x, s, g)
    assert idx.tolist() == [0, 2, 0]
    assert best[0] == second[0] == 3.0           # exact tie reported with zero gap
    idx_p, best_p, _ = o.assign(x, s, None)      # plain projection x.s
    assert idx_p.tolist() == [0, 2, 0] and best_p.tolist() == [2.0, 3.0, 1.0]


# ---------------------------------------------------------------- shape update (Eq. 6, 7)
def test_shapes_unit_norm_and_maximise_angular_objective():
    rng = np.random.default_rng(1)
    N, d, K = 3000, 8, 16
    x = rng.standard_normal((N, d)).astype(np.float32) * np.exp(rng.standard_normal((N, 1))).astype(np.float32)
    w = np.exp(rng.standard_normal(N)).astype(np.float32)
    f = o.fit_stage(x, w, K, 5, seed=3)
    s, g, idx = f["shapes"], f["gains"], f["idx_last"]
    assert np.abs(np.linalg.norm(s.astype(np.float64), axis=1) - 1).max() <= 1e-6
    assert (g >= 0).all()
    # after one more update from idx, s_k maximises sum_i w_i y_i.s over the unit sphere
    s2, g2, _, cnt = o.update(x, w, idx, s, g)
    y = x.astype(np.float64) / (np.linalg.norm(x.astype(np.float64), axis=1, keepdims=True) + 1e-12)
    for k in range(K):
        m = idx == k
        if cnt[k] == 0:
            continue
        obj = lambda u: float((w[m, None] * y[m] * u[None]).sum())
        top = obj(s2[k].astype(np.float64))
        for _ in range(20):
            assert top >= obj(_unit(rng.standard_normal(d))) - 1e-9
        b = (w[m, None] * y[m]).sum(0)
        np.testing.assert_allclose(s2[k], b / np.linalg.norm(b), atol=1e-7)


# ---------------------------------------------------------------- gain update (Eq. 8)
def test_gain_is_closed_form_minimiser_and_clamps_at_zero():
    rng = np.random.default_rng(2)
    N, d, K = 2000, 4, 6
    x = rng.standard_normal((N, d)).astype(np.float32)
    w = np.exp(rng.standard_normal(N)).astype(np.float32)
    s, g = _rand_codebook(rng, K, d)
    idx = rng.integers(0, K, N).astype(np.int32)
    # force cluster 0 to have negative mean projection: members are points opposite to s_0
    m0 = idx == 0
    x[m0] = (-np.abs(rng.standard_normal((m0.sum(), 1))) * s[0][None]).astype(np.float32)
    s_same, g_new, _, _ = o.update(x, w, idx, s, g, shapes_too=False)
    assert np.array_equal(s_same, s)
    assert g_new[0] == 0.0
    J = o.wdist(x, w, idx, s, g_new)
    for k in range(1, K):
        m = idx == k
        want = max(0.0, float((w[m] * (x[m].astype(np.float64) @ s[k].astype(np.float64))).sum() / w[m].sum()))
        assert abs(g_new[k] - want) <= 1e-6 * max(1, want)
        for h in (1e-2, -1e-2):
            gp = g_new.copy()
            gp[k] = max(0.0, gp[k] + h)
            assert o.wdist(x, w, idx, s, gp) >= J - 1e-9 * J
    # clamp: with g_0 = 0 any positive gain is worse
    gp = g_new.copy(); gp[0] = 1e-2
    assert o.wdist(x, w, idx, s, gp) > J


# ---------------------------------------------------------------- weighted reading (c-W)
def test_integer_weights_equal_replicated_rows_and_weight_scale_invariance():
    rng = np.random.default_rng(3)
    N, d, K = 600, 8, 8
    x = (rng.standard_normal((N, d)) * np.exp(0.5 * rng.standard_normal((N, 1)))).astype(np.float32)
    w = rng.integers(1, 4, N).astype(np.float32)
    s0, g0 = _rand_codebook(rng, K, d)
    idx, _, _ = o.assign(x, s0, g0)
    s_w, g_w, _, _ = o.update(x, w, idx, s0, g0)
    rep = np.repeat(np.arange(N), w.astype(int))
    s_r, g_r, _, _ = o.update(x[rep], None, idx[rep], s0, g0)
    np.testing.assert_allclose(s_w, s_r, atol=1e-7)
    np.testing.assert_allclose(g_w, g_r, rtol=1e-6)
    assert abs(o.wdist(x, w, idx, s_w, g_w) - o.wdist(x[rep], None, idx[rep], s_w, g_w)) <= 1e-9 * N
    # scaling every weight by 2 (exact in binary fp): identical codebook bits, J doubles
    fa = o.fit_stage(x, w, K, 6, seed=11)
    fb = o.fit_stage(x, 2 * w, K, 6, seed=11)
    assert np.array_equal(fa["shapes"], fb["shapes"]) and np.array_equal(fa["gains"], fb["gains"])
    np.testing.assert_allclose(fb["J_assign"], 2 * fa["J_assign"], rtol=1e-14)


# ---------------------------------------------------------------- whole update: reductions to known algorithms
def _lloyd(x, w, mu, iters):
    """Textbook weighted Lloyd K-means (float64); returns centroids after `iters` iterations."""
    x = x.astype(np.float64); mu = mu.astype(np.float64).copy()
    for _ in range(iters):
        a = ((x[:, None] - mu[None]) ** 2).sum(-1).argmin(1)
        for k in range(len(mu)):
            m = a == k
            if m.any():
                mu[k] = (w[m, None] * x[m]).sum(0) / w[m].sum()
    return mu


def test_equal_norm_rows_reduce_to_weighted_lloyd_kmeans():
    """If all ||x_i|| are equal, sum w y is proportional to sum w x, so g_k s_k is the weighted mean."""
    from sklearn.cluster import KMeans
    rng = np.random.default_rng(4)
    N, d, K, iters = 1500, 4, 6, 7
    x = (3.0 * _unit(rng.standard_normal((N, d)) + np.array([1.5, 0, 0, 0]))).astype(np.float32)
    x = (3.0 * _unit(x.astype(np.float64))).astype(np.float32)
    w = np.exp(0.5 * rng.standard_normal(N)).astype(np.float32)
    ids = o.init_ids(x, K, 7)
    s = _unit(x[ids].astype(np.float64)).astype(np.float32)
    a0, _, _ = o.assign(x, s, None)
    _, g, _, _ = o.update(x, w, a0, s, np.zeros(K, np.float32), shapes_too=False)
    mu0 = g[:, None].astype(np.float64) * s.astype(np.float64)
    # oracle trajectory, step by step
    so, go = s, g
    for _ in range(iters):
        a, _, _ = o.assign(x, so, go)
        so, go, n_empty, _ = o.update(x, w, a, so, go)
        assert n_empty == 0
    mu_or = go[:, None].astype(np.float64) * so.astype(np.float64)
    np.testing.assert_allclose(mu_or, _lloyd(x, w.astype(np.float64), mu0, iters), atol=2e-5)
    km = KMeans(n_clusters=K, init=mu0, n_init=1, max_iter=iters, tol=0.0, algorithm="lloyd")
    km.fit(x.astype(np.float64), sample_weight=w.astype(np.float64))
    np.testing.assert_allclose(mu_or, km.cluster_centers_, atol=2e-5)
    # and the same through fit_stage
    f = o.fit_stage(x, w, K, iters, seed=7)
    np.testing.assert_allclose(f["gains"][:, None] * f["shapes"], mu_or, atol=1e-6)
    assert (np.diff(f["J_assign"]) <= 1e-9 * f["J_assign"][0]).all()      # Lloyd is monotone


def test_K1_closed_form():
    rng = np.random.default_rng(6)
    x = (rng.standard_normal((400, 8)) + 0.7).astype(np.float32)
    w = np.exp(rng.standard_normal(400)).astype(np.float32)
    f = o.fit_stage(x, w, 1, 3, seed=1)
    xd, wd = x.astype(np.float64), w.astype(np.float64)
    y = xd / (np.linalg.norm(xd, axis=1, keepdims=True) + 1e-12)
    s = _unit((wd[:, None] * y).sum(0))
    g = max(0.0, float((wd * (xd @ s.astype(np.float32).astype(np.float64))).sum() / wd.sum()))
    np.testing.assert_allclose(f["shapes"][0], s, atol=1e-7)
    assert abs(f["gains"][0] - g) <= 1e-6 * g
    assert f["iters_run"] == 2                      # assignments cannot change with K = 1


def test_hand_computed_nonmonotone_example():
    """no monotone-decrease guarantee.  Golden values derived by hand from Eq. 6-8."""
    gold = {}
    for line in (GOLD / "nonmonotone_example.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        gold[k] = [float(t) for t in v]
    x = np.array([[100, 0]] + [[0, 1]] * 10, np.float32)
    s0 = np.array([gold["s0"]], np.float32)
    a = np.zeros(11, np.int32)
    _, g0, _, _ = o.update(x, None, a, s0, np.zeros(1, np.float32), shapes_too=False)
    assert abs(g0[0] - gold["g0"][0]) < 1e-6
    assert abs(o.wdist(x, None, a, s0, g0) - gold["J0"][0]) < 1e-3      # g0 is fp32-rounded
    s1, g1, _, _ = o.update(x, None, a, s0, g0)
    np.testing.assert_allclose(s1[0], gold["s1"], atol=1e-7)
    assert abs(g1[0] - gold["g1"][0]) < 1e-6
    J1 = o.wdist(x, None, a, s1, g1)
    assert abs(J1 - gold["J1"][0]) < 1e-3
    assert J1 > gold["J0"][0] + 800                  # the distortion ROSE
    y = x / np.linalg.norm(x, axis=1, keepdims=True)
    assert abs((y @ s0[0]).sum() - gold["ang0"][0]) < 1e-6
    assert abs((y.astype(np.float64) @ s1[0].astype(np.float64)).sum() - gold["ang1"][0]) < 1e-5


# ---------------------------------------------------------------- provable monotone pieces (reading c-M)
def test_assignment_and_gain_steps_never_increase_J():
    d0 = inputs.make(0)
    x, K = d0["x"][0], 16
    w = np.exp(np.random.default_rng(9).standard_normal(len(x))).astype(np.float32)
    ids = o.init_ids(x, K, 0)
    s = _unit(x[ids].astype(np.float64)).astype(np.float32)
    a, _, _ = o.assign(x, s, None)
    _, g, _, _ = o.update(x, w, a, s, np.zeros(K, np.float32), shapes_too=False)
    for _ in range(6):
        J_before = o.wdist(x, w, a, s, g)
        a_new, _, _ = o.assign(x, s, g)
        J_assign = o.wdist(x, w, a_new, s, g)
        assert J_assign <= J_before * (1 + 1e-12)                  # (i) assignment step
        s_new, g_new, _, _ = o.update(x, w, a_new, s, g)
        _, g_only, _, _ = o.update(x, w, a_new, s_new, g, shapes_too=False)
        assert np.array_equal(g_only, g_new)                       # Eq. 8 uses the UPDATED shape
        J_shape_oldgain = o.wdist(x, w, a_new, s_new, g)
        assert o.wdist(x, w, a_new, s_new, g_new) <= J_shape_oldgain * (1 + 1e-7)   # (ii) gain step
        a, s, g = a_new, s_new, g_new


@pytest.mark.parametrize("cfg,T", [(0, None), (1, 256), (2, 256)])
def test_J_non_increasing_on_baseline_generators(cfg, T):
    """BASELINE.json asks for this check; it is NOT a theorem -- asserted only on
    these generators, where it holds empirically (reading c-M)."""
    dd = inputs.make(cfg, T=T)
    c = dd["config"]
    rows = o.rows_of(dd["x"], c.d)[0]
    M = c.hd // c.d
    w = None if dd["w"] is None else np.repeat(dd["w"], M)
    K = c.K if cfg == 0 else 64
    f = o.fit_stage(rows, w, K, 10, seed=0)
    J = f["J_assign"]
    assert (np.diff(J) <= 1e-9 * J[0]).all(), J


# ---------------------------------------------------------------- equivariances, idempotence
def test_scale_by_two_is_bit_exact():
    dd = inputs.make(0)
    x = dd["x"][0][:1500]
    fa = o.fit_stage(x, None, 16, 8, seed=0)
    fb = o.fit_stage(2 * x, None, 16, 8, seed=0)
    assert np.array_equal(fa["idx_last"], fb["idx_last"])
    assert np.array_equal(fa["shapes"], fb["shapes"])
    assert np.array_equal(2 * fa["gains"], fb["gains"])


def test_rotation_and_permutation_equivariance():
    rng = np.random.default_rng(8)
    N, d, K = 1200, 8, 12
    x = (rng.standard_normal((N, d)) * np.exp(0.5 * rng.standard_normal((N, 1)))).astype(np.float64)
    q, _ = np.linalg.qr(rng.standard_normal((d, d)))
    s0, g0 = _rand_codebook(rng, K, d)
    a1, b1, s1_ = o.assign(x, s0, g0)
    xq = (x @ q.T).astype(np.float32)
    sq = (s0.astype(np.float64) @ q.T).astype(np.float32)
    a2, _, _ = o.assign(xq, sq, g0)
    safe = (b1 - s1_) > 1e-4                       # fp32 rounding of rotated operands can flip true near-ties
    assert np.array_equal(a1[safe], a2[safe])
    su, gu, _, _ = o.update(x.astype(np.float32), None, a1, s0, g0)
    sv, gv, _, _ = o.update(xq, None, a1, sq, g0)
    np.testing.assert_allclose(su.astype(np.float64) @ q.T, sv, atol=5e-6)
    np.testing.assert_allclose(gu, gv, rtol=2e-5)
    # permutation of rows: same sums up to double rounding
    p = rng.permutation(N)
    xf = x.astype(np.float32)
    sp, gp, _, _ = o.update(xf[p], None, a1[p], s0, g0)
    np.testing.assert_allclose(su, sp, atol=1e-7)
    np.testing.assert_allclose(gu, gp, rtol=1e-6)


def test_update_after_convergence_is_exact_noop():
    dd = inputs.make(0)
    x = dd["x"][0][:800]
    f = o.fit_stage(x, None, 8, 200, seed=2)
    assert f["iters_run"] < 200 and f["changed"][-1] == 0
    a, _, _ = o.assign(x, f["shapes"], f["gains"])
    assert np.array_equal(a, f["idx_last"])
    s2, g2, _, _ = o.update(x, None, a, f["shapes"], f["gains"])
    assert np.array_equal(s2, f["shapes"]) and np.array_equal(g2, f["gains"])
    # hence "run exactly iters" == "break early" (reading c-C)
    f2 = o.fit_stage(x, None, 8, f["iters_run"] - 1, seed=2)
    assert np.array_equal(f2["shapes"], f["shapes"]) and np.array_equal(f2["gains"], f["gains"])


def test_empty_cluster_and_zero_direction_safeguards():
    """empty cluster keeps (g, s); near-zero mean direction keeps s."""
    x = np.array([[1, 0], [-1, 0], [0, 2], [0, 0]], np.float32)
    s = np.array([[0.6, 0.8], [0, 1], [1, 0]], np.float32)
    g = np.array([0.5, 1.0, 7.0], np.float32)
    idx = np.array([0, 0, 1, 1], np.int32)              # cluster 2 empty; cluster 0 has y's that cancel
    s2, g2, n_empty, cnt = o.update(x, None, idx, s, g)
    assert n_empty == 1 and cnt.tolist() == [2, 2, 0]
    assert np.array_equal(s2[2], s[2]) and g2[2] == g[2]
    assert np.array_equal(s2[0], s[0]) and g2[0] == 0.0  # direction kept, gain = max(0, mean proj = 0)
    np.testing.assert_allclose(s2[1], [0, 1], atol=1e-7)  # zero row contributes 0 to B but counts in W
    assert abs(g2[1] - 1.0) < 1e-7                       # (2 + 0)/2


# ---------------------------------------------------------------- RQ / decode
def test_rq_identities_prefix_property_and_energy():
    dd = inputs.make(1, T=96)
    c = dd["config"]
    x, w = dd["x"][:2], dd["w"]
    K, S = 32, 3
    out = o.gsrq_fit_encode(x, w, c.d, K, S, 6, seed=0)
    rows = o.rows_of(x, c.d)
    M = c.hd // c.d
    w_rows = np.repeat(w, M).astype(np.float64)
    for g_ in range(2):
        rec = o.decode_rows(out["codes"][:, g_], out["shapes"][g_], out["gains"][g_])
        # x = sum_s c^(s)[a^(s)] + r^(S) to fp32 rounding
        np.testing.assert_allclose(rec + out["residual"][g_], rows[g_], atol=2e-5 * np.abs(rows[g_]).max())
        # stage-order fp32 sum written out with numpy fp32 ops
        cw = (out["gains"][g_][:, :, None] * out["shapes"][g_]).astype(np.float32)
        acc = cw[0][out["codes"][0, g_]]
        for st in range(1, S):
            acc = (acc + cw[st][out["codes"][st, g_]]).astype(np.float32)
        assert np.array_equal(acc, rec)
        # prefix decode == decode of truncated codes
        assert np.array_equal(o.decode_rows(out["codes"][:, g_], out["shapes"][g_], out["gains"][g_], 2),
                              o.decode_rows(out["codes"][:2, g_], out["shapes"][g_, :2], out["gains"][g_, :2]))
        # weighted residual energy is non-increasing stage by stage on the fit set (reading c-N)
        e = [float((w_rows * (rows[g_].astype(np.float64) ** 2).sum(1)).sum())]
        r = rows[g_].copy()
        for st in range(S):
            _, r, _, _ = o.encode_stage(r, out["shapes"][g_, st], out["gains"][g_, st])
            e.append(float((w_rows * (r.astype(np.float64) ** 2).sum(1)).sum()))
        assert all(e[i + 1] <= e[i] * (1 + 1e-9) for i in range(S)), e
    # greedy prefix property: first 2 stages of the 3-stage run == a 2-stage run
    out2 = o.gsrq_fit_encode(x, w, c.d, K, 2, 6, seed=0)
    assert np.array_equal(out2["shapes"], out["shapes"][:, :2]) and np.array_equal(out2["codes"], out["codes"][:2])
    # encode() with the fitted codebooks reproduces the codes
    codes, res, _, _ = o.encode(x, out["shapes"], out["gains"], c.d)
    assert np.array_equal(codes, out["codes"]) and np.array_equal(res, out["residual"])


def test_bitrates_match_paper():
    for line in (GOLD / "bitrates.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        R, K, D, bpa = line.split()
        assert abs(int(R) * math.log2(int(K)) / int(D) - float(bpa)) < 1e-12


def test_bf16_cast_matches_torch_round_to_nearest_even():
    import torch
    rng = np.random.default_rng(10)
    x = np.concatenate([rng.standard_normal(20000) * np.exp(4 * rng.standard_normal(20000)),
                        [0.0, -0.0, 1.0, 1.00390625, 1.01171875, 3.3895314e38, 1e-40, -1e-45]]).astype(np.float32)
    bits = o.f32_to_bf16_bits(x)
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(bits, want)
    val, b = o.decode(np.zeros((1, 1, 8), np.uint8), np.ones((1, 1, 1, 16), np.float32) * 0.25,
                      np.full((1, 1, 1), 1.00390625 * 4, np.float32), hd=128)
    assert val.shape == (1, 1, 128) and np.all(val == 1.0) and b.dtype == np.uint16   # tie -> even


def test_fit_subset_equals_fit_on_gathered_rows():
    dd = inputs.make(1, T=128)
    c = dd["config"]
    x, w = dd["x"][:1], dd["w"]
    ft = inputs.fit_sample(1, 128, 40, 77)
    out = o.gsrq_fit_encode(x, w, c.d, 16, 1, 4, seed=0, fit_tokens=ft)
    M = c.hd // c.d
    rows = o.rows_of(x, c.d)[0].reshape(128, M, c.d)[ft[0]].reshape(-1, c.d)
    f = o.fit_stage(rows, np.repeat(w[ft[0]], M), 16, 4, seed=0, group=0, G=1, stage=0)
    assert np.array_equal(out["shapes"][0, 0], f["shapes"])
    assert out["codes"].shape == (1, 1, 128 * M)
