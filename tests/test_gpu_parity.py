"""GPU parity tests: the CUDA path (through the C-ABI binding) vs the CPU oracle, element by
element, on the same seeded inputs.  Run with `-m gpu` on a B200.

Criteria (BASELINE.json north_star): (a) code indices bit-exact except where the oracle's top-2
score gap < 1e-5*||x||; (b) codewords and gains within 1e-4 absolute; (c) final weighted
distortion within 1e-4 relative.  Two modes: lock-step and free-running.
"""
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


def _non_exempt_mismatches(got_codes, ref, rows_norm):
    """criterion (a): mismatches where the oracle's top-2 gap >= 1e-5 * ||row||."""
    gap = ref["best"] - ref["second"]
    return int(((got_codes != ref["codes"]) & (gap >= 1e-5 * rows_norm[None])).sum())


def _wdist_final(residual, w_rows):
    return float((w_rows * (residual.astype(np.float64) ** 2).sum(-1)).sum())


def _check_free_running(dd, K, S, iters, dtype, **kw):
    c = dd["config"]
    x, w = dd["x"], dd["w"]
    ref = o.gsrq_fit_encode(x, w, c.d, K, S, iters, seed=0, fit_tokens=dd.get("fit_tokens"))
    got = gpu_gsrq(x, w, c.d, K, S, iters, seed=0, dtype=dtype, fit_tokens=dd.get("fit_tokens"), **kw)
    G = x.shape[0]
    M = c.hd // c.d
    # (b) codebooks
    assert np.abs(got["shapes"] - ref["shapes"]).max() <= 1e-4
    assert np.abs(got["gains"] - ref["gains"]).max() <= 1e-4
    # (a) codes
    bad = 0
    r = o.rows_of(x, c.d).copy()
    for st in range(S):
        n_st = np.linalg.norm(r.astype(np.float64), axis=-1)
        gap = ref["best"][st] - ref["second"][st]
        bad += int(((got["codes"][st] != ref["codes"][st]) & (gap >= 1e-5 * n_st)).sum())
        for g_ in range(G):
            _, r[g_], _, _ = o.encode_stage(r[g_], ref["shapes"][g_, st], ref["gains"][g_, st])
    assert bad == 0, f"{bad} non-exempt code mismatches"
    # (c) final weighted distortion (from each side's own residual) + per-iteration J + stats
    for g_ in range(G):
        w_rows = np.ones(r.shape[1]) if w is None else np.repeat(w, M).astype(np.float64)
        jr, jg = _wdist_final(ref["residual"][g_], w_rows), _wdist_final(got["residual"][g_], w_rows)
        assert abs(jr - jg) <= 1e-4 * jr
        for st in range(S):
            s_ref, s_got = ref["stats"][g_][st], stats_np(got["stats"][st], g_)
            assert s_got["iters_run"] == s_ref["iters_run"]
            np.testing.assert_allclose(s_got["J"], s_ref["J_assign"], rtol=1e-4)
            assert np.array_equal(s_got["changed"], s_ref["changed"])
            assert s_got["n_empty_last"] == s_ref["n_empty_last"]
    return got, ref


def test_cfg0_free_running_fit_encode_decode():
    dd = inputs.make(0)
    c = dd["config"]
    got, ref = _check_free_running(dd, c.K, c.S, c.iters, "f32")
    # in practice the trajectories are identical (fp64 reduction + exact arg-max)
    assert np.array_equal(got["codes"], ref["codes"])
    dec = gpu_decode(got["codes_dev"], got["cb"], c.S, c.G, c.T, c.hd, c.d, dtype="f32")
    want, _ = o.decode(got["codes"], got["shapes"], got["gains"], c.hd, bf16=False)
    assert np.array_equal(dec, want)
    # decode(encode(x)) + residual == x to fp32 rounding
    np.testing.assert_allclose(dec.reshape(got["residual"].shape) + got["residual"], o.rows_of(dd["x"], c.d), atol=1e-5)


@pytest.mark.parametrize("cfg,kind,T,K,S,iters", [(1, "k", 160, 256, 2, 6), (2, "v", 192, 256, 1, 6),
                                                  (1, "k", 67, 100, 3, 4)])
def test_bf16_free_running_small(cfg, kind, T, K, S, iters):
    """cfg 1/2 generators at sizes the oracle finishes in seconds; T*M spans several 2048-row chunks
    only partly (ragged tail) and K=100 exercises a non-power-of-two codebook."""
    dd = inputs.make(cfg, kind=kind, T=T)
    _check_free_running(dd, K, S, iters, "bf16")


def test_bf16_free_running_multi_chunk_with_fit_subset_and_head_inner():
    dd = inputs.make(4, kind="k", T=1024)           # n_fit = 64 tokens/head -> 512 fit rows/head
    dd["fit_tokens"] = inputs.fit_sample(8, 1024, 320, inputs.seed_of(4, "fit"))   # 2560 rows: 2 chunks, ragged
    got, ref = _check_free_running(dd, 64, 2, 5, "bf16", head_inner=True, pass_residual=False)
    c = dd["config"]
    dec = gpu_decode(got["codes_dev"], got["cb"], 2, c.G, 1024, c.hd, c.d, dtype="bf16", head_inner=True)
    want, _ = o.decode(got["codes"], got["shapes"], got["gains"], c.hd, bf16=True)
    assert np.array_equal(dec, want)


def test_lock_step_cfg1_head(B):
    """Per iteration: oracle codebook -> one GPU assignment; oracle assignment -> one GPU update.
    Zero non-exempt index mismatches and codebooks within 1e-4 at every step."""
    dd = inputs.make(1, T=512)
    c = dd["config"]
    x_np, w_np = dd["x"][:2], dd["w"]
    G, K, d, M = 2, 256, c.d, c.hd // c.d
    x = to_device(x_np, "bf16")
    view = B.view_of(x, d)
    w = torch.from_numpy(w_np).cuda()
    ws = B.workspace(view, K, 1, 0)
    rows = o.rows_of(x_np, d)
    w_rows = np.repeat(w_np, M)
    shapes = torch.zeros(G, 1, K, d, device="cuda")
    gains = torch.zeros(G, 1, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    idx_dev = torch.zeros(G, rows.shape[1], dtype=torch.uint8, device="cuda")
    # init ids
    ids_dev = torch.zeros(G, K, dtype=torch.int64, device="cuda")
    B.gsrq_init_ids(x, view, None, None, K, 0, 0, ids_dev, ws)
    ids = ids_dev.cpu().numpy()
    s_or = np.zeros((G, K, d), np.float32); g_or = np.zeros((G, K), np.float32)
    for g_ in range(G):
        want = o.init_ids(rows[g_], K, 0, group=g_, G=G, stage=0)
        assert np.array_equal(ids[g_], want)
        r = rows[g_][want].astype(np.float64)
        s_or[g_] = (r / np.linalg.norm(r, axis=1, keepdims=True)).astype(np.float32)
    nrm = np.linalg.norm(rows.astype(np.float64), axis=-1)
    for t in range(0, 5):
        # GPU assignment with the ORACLE's codebook
        shapes.copy_(torch.from_numpy(s_or[:, None]).cuda()); gains.copy_(torch.from_numpy(g_or[:, None]).cuda())
        B.gsrq_assign(x, view, None, cb, 0, 1 if t == 0 else 0, idx_dev, ws)
        idx_gpu = idx_dev.cpu().numpy()
        for g_ in range(G):
            a, best, second = o.assign(rows[g_], s_or[g_], None if t == 0 else g_or[g_])
            mism = (idx_gpu[g_] != a)
            assert not (mism & ((best - second) >= 1e-5 * nrm[g_])).any()
            assert not mism.any()           # exact refine: identical, not merely within the exemption
            # GPU update from the ORACLE's assignment
            idx_dev[g_].copy_(torch.from_numpy(a.astype(np.uint8)).cuda())
        B.gsrq_update(x, view, None, w, 0, idx_dev, cb, 0, t > 0, ws)
        s_gpu, g_gpu = shapes.cpu().numpy()[:, 0], gains.cpu().numpy()[:, 0]
        for g_ in range(G):
            a, _, _ = o.assign(rows[g_], s_or[g_], None if t == 0 else g_or[g_])
            s_or[g_], g_or[g_], _, _ = o.update(rows[g_], w_rows, a, s_or[g_], g_or[g_], shapes_too=t > 0)
        assert np.abs(s_gpu - s_or).max() <= 1e-4 and np.abs(g_gpu - g_or).max() <= 1e-4
        assert np.abs(s_gpu - s_or).max() <= 1e-7          # fp64 sums: same fp32 codebook up to 1 ulp


def test_encode_stage_ranges_residual_and_prefix_decode(B):
    dd = inputs.make(1, T=96)
    c = dd["config"]
    x_np = dd["x"]
    S, K = 3, 64
    got = gpu_gsrq(x_np, dd["w"], c.d, K, S, 3, dtype="bf16")
    x, view, cb, ws = got["x"], got["view"], got["cb"], got["ws"]
    G, Ng = c.G, 96 * (c.hd // c.d)
    # fused [0,S) == stage by stage
    codes_f = torch.zeros(S, G, Ng, dtype=torch.uint8, device="cuda")
    res_f = torch.zeros(G, Ng, c.d, device="cuda")
    B.gsrq_encode(x, view, cb, 0, S, codes_f, res_f, ws)
    assert torch.equal(codes_f, got["codes_dev"])
    assert np.array_equal(res_f.cpu().numpy(), got["residual"])
    # oracle, fixed codebooks
    codes_o, res_o, _, _ = o.encode(x_np, got["shapes"], got["gains"], c.d)
    assert np.array_equal(codes_o, got["codes"]) and np.array_equal(res_o, got["residual"])
    # resume at stage 2 from planes 0-1 (earlier planes are read)
    codes_r = codes_f.clone(); codes_r[2].zero_()
    res_r = torch.zeros_like(res_f)
    B.gsrq_encode(x, view, cb, 2, 3, codes_r, res_r, ws)
    assert torch.equal(codes_r, codes_f) and torch.equal(res_r, res_f)
    # prefix decode in bf16 and fp32
    for n in range(0, S + 1):
        dec = gpu_decode(codes_f, cb, n, G, 96, c.hd, c.d, dtype="bf16")
        want, _ = o.decode(got["codes"], got["shapes"], got["gains"], c.hd, S_used=n, bf16=True)
        assert np.array_equal(dec, want), n
    dec32 = gpu_decode(codes_f, cb, S, G, 96, c.hd, c.d, dtype="f32")
    want32, _ = o.decode(got["codes"], got["shapes"], got["gains"], c.hd, bf16=False)
    assert np.array_equal(dec32, want32)


def test_fit_stage_residual_null_equals_residual_given():
    dd = inputs.make(2, T=128)
    c = dd["config"]
    a = gpu_gsrq(dd["x"], dd["w"], c.d, 32, 3, 4, dtype="bf16", pass_residual=True)
    b = gpu_gsrq(dd["x"], dd["w"], c.d, 32, 3, 4, dtype="bf16", pass_residual=False)
    for k in ("shapes", "gains", "codes", "residual"):
        assert np.array_equal(a[k], b[k]), k


def test_run_to_run_bit_identical():
    dd = inputs.make(1, T=300)
    c = dd["config"]
    a = gpu_gsrq(dd["x"], dd["w"], c.d, 256, 2, 5, dtype="bf16")
    b = gpu_gsrq(dd["x"], dd["w"], c.d, 256, 2, 5, dtype="bf16")
    for k in ("shapes", "gains", "codes", "residual"):
        assert np.array_equal(a[k], b[k]), k
    for st in range(2):
        for g_ in range(c.G):
            assert np.array_equal(stats_np(a["stats"][st], g_)["J"], stats_np(b["stats"][st], g_)["J"])


def test_degenerate_and_edge_inputs(B):
    # all-zero tensor: no K distinct non-zero rows -> GSRQ_EDEGENERATE
    x = torch.zeros(1, 64, 16, device="cuda")
    view = B.view_of(x, 8)
    shapes = torch.zeros(1, 1, 16, 8, device="cuda"); gains = torch.zeros(1, 1, 16, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, 16, 1)
    with pytest.raises(B.GsrqError) as e:
        B.gsrq_fit_stage(x, view, None, 0, None, cb, 0, None, 3, 0, ws)
    assert e.value.code == -5
    # fewer rows than K
    x2 = torch.randn(1, 4, 8, device="cuda")
    with pytest.raises(B.GsrqError):
        B.gsrq_fit_stage(x2, B.view_of(x2, 8), None, 0, None, cb, 0, None, 3, 0, B.workspace(B.view_of(x2, 8), 16, 1))
    # workspace too small
    with pytest.raises(B.GsrqError) as e:
        B.gsrq_encode(x, view, cb, 0, 1, torch.zeros(1, 1, 128, dtype=torch.uint8, device="cuda"), None, ws[:256])
    assert e.value.code == -3
    # zero rows and zero-gain clusters encode to something valid; K = 1
    rng = np.random.default_rng(0)
    xn = rng.standard_normal((1, 40, 16)).astype(np.float32); xn[0, ::5] = 0
    got = gpu_gsrq(xn, None, 8, 1, 1, 3, dtype="f32")
    ref = o.gsrq_fit_encode(xn, None, 8, 1, 1, 3)
    assert np.array_equal(got["codes"], ref["codes"]) and np.abs(got["shapes"] - ref["shapes"]).max() < 1e-6
    assert stats_np(got["stats"][0], 0)["iters_run"] == ref["stats"][0][0]["iters_run"] == 2


@pytest.mark.parametrize("d,hd", [(8, 16), (16, 128), (128, 128)])
def test_fit_status_reports_what_an_asynchronous_fit_cannot(B, d, hd):
    """gsrq_fit_stage(stats = NULL) returns GSRQ_OK before the kernels have run; gsrq_fit_status reads the per-group error words
    afterwards (include/gsrq.h): a group of all-zero rows is degenerate (GSRQ_EDEGENERATE), a healthy fit reports GSRQ_OK."""
    G, T, K = 2, 512, 16
    x = torch.randn(G, T, hd, device="cuda", generator=torch.Generator(device="cuda").manual_seed(3))
    if d == 16:
        x = x.bfloat16()   # the persistent tensor-core fit kernel
    shapes = torch.zeros(G, 1, K, d, device="cuda"); gains = torch.zeros(G, 1, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    view = B.view_of(x, d)
    ws = B.workspace(view, K, 1)
    B.gsrq_fit_stage(x, view, None, 0, None, cb, 0, None, 3, 0, ws, want_stats=False)
    B.gsrq_fit_status(ws, view, K, 1)          # healthy: no error
    assert torch.isfinite(shapes).all() and (shapes.norm(dim=-1) - 1).abs().max() < 1e-5
    x[1].zero_()                               # group 1 has no non-zero row
    B.gsrq_fit_stage(x, view, None, 0, None, cb, 0, None, 3, 0, ws, want_stats=False)   # asynchronous: cannot know yet
    with pytest.raises(B.GsrqError) as e:
        B.gsrq_fit_status(ws, view, K, 1)
    assert e.value.code == -5
