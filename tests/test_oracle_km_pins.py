"""Pins of the K-means baseline and the quality metrics of oracle/km_oracle.c (section 6.1, :200-212; section 4) against
things other than itself: scikit-learn's Lloyd K-means from the same initial centroids, numpy's own formulas, closed forms and
the inequalities the paper states.  CPU only."""
import numpy as np
import pytest

from oracle import gsrq_oracle as o


def _rows(N, d, seed, scale=True):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((N, d))
    if scale:
        x *= np.exp(0.5 * rng.standard_normal(N))[:, None]
    return x.astype(np.float32)


def test_km_assignment_is_brute_force_nearest_centroid_with_lowest_index_ties():
    x = _rows(300, 6, 1)
    mu = _rows(17, 6, 2)
    mu[9] = mu[3]                                   # duplicate centroid: the lower index must win
    idx, best = o.km_assign(x, mu)
    d2 = ((x[:, None, :].astype(np.float64) - mu[None].astype(np.float64)) ** 2).sum(-1)
    assert np.array_equal(idx, d2.argmin(1))
    np.testing.assert_allclose(best, d2.min(1), rtol=1e-12)
    assert not (idx == 9).any()


def test_km_update_is_the_weighted_mean_and_equals_replicated_rows():
    x = _rows(200, 5, 3)
    rng = np.random.default_rng(4)
    idx = rng.integers(0, 7, 200).astype(np.int32)
    idx[idx == 5] = 4                               # cluster 5 is empty: keeps its centroid
    w = rng.integers(1, 4, 200).astype(np.float32)
    mu0 = _rows(7, 5, 5)
    mu, ne = o.km_update(x, w, idx, mu0)
    assert ne == 1 and np.array_equal(mu[5], mu0[5])
    for k in (0, 1, 2, 3, 4, 6):
        m = idx == k
        want = (w[m, None].astype(np.float64) * x[m].astype(np.float64)).sum(0) / w[m].astype(np.float64).sum()
        np.testing.assert_allclose(mu[k], want.astype(np.float32), rtol=0, atol=1e-7)
    rep = np.repeat(np.arange(200), w.astype(int))   # integer weights == physically replicated rows
    mu_r, _ = o.km_update(x[rep], None, idx[rep], mu0)
    np.testing.assert_allclose(mu_r, mu, atol=1e-6)


def test_km_fit_matches_scikit_learn_lloyd_from_the_same_init():
    from sklearn.cluster import KMeans
    x = _rows(1500, 8, 6)
    w = np.exp(np.random.default_rng(7).standard_normal(1500)).astype(np.float32)
    K = 12
    ids = o.init_ids(x, K, 11)
    f = o.km_fit(x, w, K, 100, 11)
    assert f["iters_run"] < 100 and f["changed"][-1] == 0          # converged
    km = KMeans(n_clusters=K, init=x[ids].astype(np.float64), n_init=1, max_iter=300, tol=0.0, algorithm="lloyd")
    km.fit(x.astype(np.float64), sample_weight=w.astype(np.float64))
    np.testing.assert_allclose(f["mu"], km.cluster_centers_, atol=2e-5)
    assert np.array_equal(f["idx_last"], km.labels_)
    assert (np.diff(f["J_assign"]) <= 1e-9 * f["J_assign"][0]).all()   # Lloyd's distortion never increases
    np.testing.assert_allclose(f["J_assign"][-1], km.inertia_, rtol=1e-6)


def test_metrics_match_numpy_formulas_and_closed_forms():
    x = _rows(400, 7, 8)
    proto = _rows(9, 7, 9)
    idx = np.random.default_rng(10).integers(0, 9, 400).astype(np.int32)
    m = o.metrics(x, proto, idx)
    x64, p64 = x.astype(np.float64), proto.astype(np.float64)[idx]
    nx, npr = np.linalg.norm(x64, axis=1), np.linalg.norm(p64, axis=1)
    assert m["mse"] == pytest.approx(((x64 - p64) ** 2).sum(1).mean(), rel=1e-12)
    assert m["gain_err"] == pytest.approx(np.abs(nx - npr).mean(), rel=1e-12)
    assert m["cosine"] == pytest.approx(((x64 * p64).sum(1) / (nx * npr)).mean(), rel=1e-12)
    assert m["shrinkage"] == pytest.approx((npr ** 2).mean() / (nx ** 2).mean(), rel=1e-12)
    # perfect reconstruction: MSE 0, gain error 0, cosine 1, shrinkage 1; xhat = 2 x: gain error = E||x||, cosine 1, shrinkage 4
    ident = o.metrics(x, x, np.arange(400))
    assert ident["mse"] == 0.0 and ident["gain_err"] == 0.0 and ident["cosine"] == pytest.approx(1.0, abs=1e-12) and ident["shrinkage"] == pytest.approx(1.0)
    dbl = o.metrics(x, 2 * x, np.arange(400))
    assert dbl["gain_err"] == pytest.approx(nx.mean(), rel=1e-6) and dbl["cosine"] == pytest.approx(1.0, abs=1e-12) and dbl["shrinkage"] == pytest.approx(4.0, rel=1e-6)


def test_centroid_shrinkage_inequality_and_gskm_trend_on_gaussian_data():
    """PAPER.md:66 Eq. 2: the l2-optimal centroid is shorter than its members on average (shrinkage ratio < 1); PAPER.md:204-212:
    on N(0, I_D) in the under-capacity regime GSKM has higher cosine similarity and lower gain error than KM."""
    rng = np.random.default_rng(12)
    x = rng.standard_normal((2000, 64)).astype(np.float32)
    K = 16
    km = o.km_fit(x, None, K, 30, 0)
    idx_km, _ = o.km_assign(x, km["mu"])
    m_km = o.metrics(x, km["mu"], idx_km)
    assert m_km["shrinkage"] < 0.5
    gs = o.fit_stage(x, None, K, 30, 0)
    a_gs, _, _ = o.assign(x, gs["shapes"], gs["gains"])
    m_gs = o.metrics(x, gs["gains"][:, None] * gs["shapes"], a_gs)
    assert m_gs["cosine"] > m_km["cosine"] and m_gs["gain_err"] < m_km["gain_err"]
