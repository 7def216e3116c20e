"""The paper's own operating points: wide sub-vectors d = 64 / 128 / 256, K = 256, R up to 12 stages,
against the CPU oracle (which takes any d).  d = 64 / 128 go through the tcgen05 filter of k_score_tc_wide.cuh plus the
exact fp64 kernel on the undecided rows; d = 256 runs the exact kernels alone.  Run with `-m gpu` on a B200."""
import numpy as np
import pytest
import torch

from paper_2607_01065_b200.pipeline import gpu_decode, gpu_gsrq, stats_np, to_device
from oracle import gsrq_oracle as o
from paper_2607_01065_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2607_01065_b200 import binding
    return binding


def _data(kind, G, T, hd, seed):
    gen = inputs.k_like if kind == "k" else inputs.v_like
    return gen(G, T, hd, seed), inputs.token_weights(T, seed + 2)


@pytest.mark.parametrize("kind,hd,d,G,T,K,S,iters", [
    ("k", 128, 128, 2, 1500, 256, 2, 6),      # D = 128: one sub-vector per (head, token); ragged last tile
    ("v", 128, 128, 2, 1100, 100, 3, 4),      # K < 256, heavy-tailed rows, three stages
    ("k", 128, 64, 2, 700, 256, 2, 5),        # D = 64: two sub-vectors per head
    ("v", 256, 256, 2, 900, 256, 2, 4),       # D = 256 (0.375 BPA): exact kernels only
])
def test_wide_free_running_fit_encode_decode(B, kind, hd, d, G, T, K, S, iters):
    """fit -> encode -> decode on both sides from the same seed: criteria (a), (b), (c) of BASELINE.json, iterations,
    per-iteration J and changed-row counts; in practice identical trajectories."""
    x, w = _data(kind, G, T, hd, 4200 + d)
    ref = o.gsrq_fit_encode(x, w, d, K, S, iters, seed=0)
    got = gpu_gsrq(x, w, d, K, S, iters, seed=0, dtype="bf16")
    assert np.abs(got["shapes"] - ref["shapes"]).max() <= 1e-4 and np.abs(got["gains"] - ref["gains"]).max() <= 1e-4
    assert np.abs(got["shapes"] - ref["shapes"]).max() <= 1e-6      # fp64 sums on both sides: the same fp32 codebook up to an ulp
    assert np.array_equal(got["codes"], ref["codes"])
    M = hd // d
    for g_ in range(G):
        w_rows = np.repeat(w, M).astype(np.float64)
        jr = float((w_rows * (ref["residual"][g_].astype(np.float64) ** 2).sum(-1)).sum())
        jg = float((w_rows * (got["residual"][g_].astype(np.float64) ** 2).sum(-1)).sum())
        assert abs(jr - jg) <= 1e-4 * jr
        for st in range(S):
            s_ref, s_got = ref["stats"][g_][st], stats_np(got["stats"][st], g_)
            assert s_got["iters_run"] == s_ref["iters_run"]
            np.testing.assert_allclose(s_got["J"], s_ref["J_assign"], rtol=1e-4)
            assert np.array_equal(s_got["changed"], s_ref["changed"])
            assert s_got["n_empty_last"] == s_ref["n_empty_last"]
    dec = gpu_decode(got["codes_dev"], got["cb"], S, G, T, hd, d, dtype="bf16")
    want, _ = o.decode(got["codes"], got["shapes"], got["gains"], hd, bf16=True)
    assert np.array_equal(dec, want)
    assert np.array_equal(got["residual"], ref["residual"])


@pytest.mark.parametrize("S,T,prefixes", [(12, 640, (1, 5, 12)),                   # R = 12: 0.75 bits per element
                                          (16, 520, (4, 8, 12, 16)),               # R = 16: 1 bit per element
                                          (32, 2048, (4, 8, 12, 16, 20, 24, 28, 32))])   # R = 32: 2 bits per element (GSRQ_MAX_STAGES); enough rows that no stage is degenerate
def test_wide_fused_encode_many_stages_and_prefix_decode(B, S, T, prefixes):
    """R = 12 / 16 / 32 stages at D = 128 (the paper's three bit rates): one gsrq_encode of all stages with given
    codebooks equals the oracle stage by stage; prefixes decode alone; fits that re-derive their residual agree too."""
    G, hd, d, K = 2, 128, 128, 256
    x, w = _data("k", G, T, hd, 4300 + S)
    ref = o.gsrq_fit_encode(x, w, d, K, S, 2, seed=0)
    got = gpu_gsrq(x, w, d, K, S, 2, seed=0, dtype="bf16", pass_residual=False)   # fits re-derive the residual; one encode of [0, S)
    assert np.array_equal(got["codes"], ref["codes"])
    assert np.abs(got["shapes"] - ref["shapes"]).max() <= 1e-6 and np.abs(got["gains"] - ref["gains"]).max() <= 1e-5
    assert np.array_equal(got["residual"], ref["residual"])
    for n in prefixes:
        dec = gpu_decode(got["codes_dev"], got["cb"], n, G, T, hd, d, dtype="bf16")
        want, _ = o.decode(got["codes"][:n], got["shapes"][:, :n], got["gains"][:, :n], hd, bf16=True)
        assert np.array_equal(dec, want), n


def _rho(d, n_planes):
    """The filter's rho (k_score_tc_wide.cuh): accumulation budgeted at 2^-23 per step."""
    return ((9.0 if n_planes == 2 else 8.0) if d == 128 else (6.5 if n_planes == 2 else 5.5)) * 2.0 ** -17


@pytest.mark.parametrize("d,use_residual", [(128, False), (128, True), (64, True)])
def test_wide_tc_scores_within_bound(B, d, use_residual):
    """Raw tcgen05 scores at d = 64 / 128 against fp64, relative to the bound the kernel uses:
    E(g) = rho 2^-17 (2 g ||r||) + 2^-18 g^2, rho = 5.5 / 6.5 (d = 64), 8 / 9 (d = 128) for one / two operand planes."""
    G, T, hd, K = 2, 300, 128, 256
    x_np, _ = _data("k", G, T, hd, 4400 + d)
    rows = o.rows_of(x_np, d)
    res_np = None
    if use_residual:
        res_np = rows.copy()
        for g_ in range(G):
            f0 = o.fit_stage(rows[g_], None, 64, 2, seed=1)
            _, res_np[g_], _, _ = o.encode_stage(rows[g_], f0["shapes"], f0["gains"])
        rows = res_np
    s_np = np.zeros((G, 1, K, d), np.float32); g_np = np.zeros((G, 1, K), np.float32)
    for g_ in range(G):
        f = o.fit_stage(rows[g_], None, K, 2, seed=0)
        s_np[g_, 0], g_np[g_, 0] = f["shapes"], f["gains"]
    x = to_device(x_np, "bf16")
    view = B.view_of(x, d)
    res = None if res_np is None else torch.from_numpy(res_np).cuda()
    shapes, gains = torch.from_numpy(s_np).cuda(), torch.from_numpy(g_np).cuda()
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, 1, 0)
    N = rows.shape[1]
    for mode in (0, 1):
        scores = torch.zeros(G, N, 256, device="cuda")
        idx = torch.zeros(G, N, dtype=torch.uint8, device="cuda")
        B.gsrq_debug_scores(x, view, res, cb, 0, mode, scores, idx, ws)
        torch.cuda.synchronize()
        sc = scores.cpu().numpy().astype(np.float64)
        for g_ in range(G):
            r64, s64, g64 = rows[g_].astype(np.float64), s_np[g_, 0].astype(np.float64), g_np[g_, 0].astype(np.float64)
            dots = r64 @ s64.T
            exact = 2 * g64[None] * dots - g64[None] ** 2 if mode == 0 else 2 * dots
            err = np.abs(sc[g_][:, :K] - exact)
            nrm = np.linalg.norm(r64, axis=1)
            gk = g64[None] if mode == 0 else np.ones((1, K))
            rho = _rho(d, 2 if use_residual else 1)
            E = rho * 2 * gk * nrm[:, None] + (2.0 ** -18 * gk * gk if mode == 0 else 0.0)
            ratio = (err / np.maximum(E, 1e-30)).max()
            print(f"wide tc filter error / bound: {ratio:.3f} (d={d} residual={use_residual} mode={mode} g={g_})")
            assert ratio <= 0.5, f"filter error reaches {ratio:.3f} of the bound (d={d}, mode {mode}, group {g_})"
            a, _, _ = o.assign(rows[g_], s_np[g_, 0], g_np[g_, 0] if mode == 0 else None)
            assert np.array_equal(idx[g_].cpu().numpy(), a)


def test_wide_lockstep_update_and_init(B):
    """One GPU update from the oracle's assignment, and the seeded initial rows, at d = 128."""
    G, T, hd, d, K = 2, 900, 128, 128, 64
    x_np, w_np = _data("v", G, T, hd, 4500)
    rows = o.rows_of(x_np, d)
    x = to_device(x_np, "bf16")
    view = B.view_of(x, d)
    ws = B.workspace(view, K, 1, 0)
    ids = torch.zeros(G, K, dtype=torch.int64, device="cuda")
    B.gsrq_init_ids(x, view, None, None, K, 0, 7, ids, ws)
    for g_ in range(G):
        assert np.array_equal(ids[g_].cpu().numpy(), o.init_ids(rows[g_], K, 7, g_, G, 0))
    w = torch.from_numpy(w_np).cuda()
    s_np = np.zeros((G, 1, K, d), np.float32); g_np = np.zeros((G, 1, K), np.float32); a_np = np.zeros((G, T), np.uint8)
    s_want = np.zeros_like(s_np); g_want = np.zeros_like(g_np)
    for g_ in range(G):
        f = o.fit_stage(rows[g_], w_np, K, 1, seed=0)
        s_np[g_, 0], g_np[g_, 0] = f["shapes"], f["gains"]
        a, _, _ = o.assign(rows[g_], f["shapes"], f["gains"])
        a_np[g_] = a
        s2, g2, _, _ = o.update(rows[g_], w_np, a, f["shapes"].copy(), f["gains"].copy(), True)
        s_want[g_, 0], g_want[g_, 0] = s2, g2
    shapes, gains = torch.from_numpy(s_np).cuda(), torch.from_numpy(g_np).cuda()
    cb = B.codebook_of(shapes, gains)
    B.gsrq_update(x, view, None, w, 0, torch.from_numpy(a_np).cuda(), cb, 0, True, ws)
    torch.cuda.synchronize()
    assert np.abs(shapes.cpu().numpy() - s_want).max() <= 1e-7 and np.abs(gains.cpu().numpy() - g_want).max() <= 1e-6


@pytest.mark.parametrize("d", [64, 128])
def test_wide_tc_scores_within_bound_under_cancellation(B, d):
    """Adversarial input for the filter's error bound: every row is made (nearly) orthogonal to a chosen codeword, and the elements of
    rows and codewords spread over twelve binades, so that the products of a dot product are large and cancel -- the case where a
    tensor core that truncates or aligns its partial sums loses most.  The raw scores must still be within half of the bound
    E(g) (two operand planes: fp32 rows), and the arg-max must equal the exact one."""
    rng = np.random.default_rng(900 + d)
    G, T, hd, K = 2, 200, 128, 256
    M = hd // d
    N = T * M
    mag = lambda shape: np.exp2(rng.uniform(-6, 6, shape)) * rng.choice([-1.0, 1.0], shape)
    s_np = mag((G, 1, K, d))
    s_np /= np.linalg.norm(s_np, axis=-1, keepdims=True)
    s_np = s_np.astype(np.float32)
    g_np = (0.5 + np.abs(rng.standard_normal((G, 1, K)))).astype(np.float32)
    rows = mag((G, N, d))
    for g_ in range(G):   # remove the component along one codeword per row: that score is pure cancellation
        pick = s_np[g_, 0][rng.integers(0, K, N)].astype(np.float64)
        pick /= np.linalg.norm(pick, axis=1, keepdims=True)
        rows[g_] -= (rows[g_] * pick).sum(1, keepdims=True) * pick
    rows = rows.astype(np.float32)
    x = torch.zeros(G, T, hd, dtype=torch.bfloat16, device="cuda")   # the rows come in through the fp32 residual (hi + lo planes)
    view = B.view_of(x, d)
    res = torch.from_numpy(rows).cuda()
    shapes, gains = torch.from_numpy(s_np).cuda(), torch.from_numpy(g_np).cuda()
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, 1, 0)
    for mode in (0, 1):
        scores = torch.zeros(G, N, 256, device="cuda")
        idx = torch.zeros(G, N, dtype=torch.uint8, device="cuda")
        B.gsrq_debug_scores(x, view, res, cb, 0, mode, scores, idx, ws)
        torch.cuda.synchronize()
        sc = scores.cpu().numpy().astype(np.float64)
        for g_ in range(G):
            r64, s64, g64 = rows[g_].astype(np.float64), s_np[g_, 0].astype(np.float64), g_np[g_, 0].astype(np.float64)
            dots = r64 @ s64.T
            exact = 2 * g64[None] * dots - g64[None] ** 2 if mode == 0 else 2 * dots
            gk = g64[None] if mode == 0 else np.ones((1, K))
            E = _rho(d, 2) * 2 * gk * np.linalg.norm(r64, axis=1)[:, None] + (2.0 ** -18 * gk * gk if mode == 0 else 0.0)
            ratio = (np.abs(sc[g_][:, :K] - exact) / E).max()
            print(f"wide tc filter error / bound under cancellation: {ratio:.3f} (d={d} mode={mode} g={g_})")
            assert ratio <= 0.5, f"filter error reaches {ratio:.3f} of the bound (d={d}, mode {mode}, group {g_})"
            a, _, _ = o.assign(rows[g_], s_np[g_, 0], g_np[g_, 0] if mode == 0 else None)
            assert np.array_equal(idx[g_].cpu().numpy(), a)
